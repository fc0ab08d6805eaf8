"""GPU parity of SSD-type pool devices (KV-passthrough; Algorithm 1 l.20-21) against the CPU oracle.

There is no NVMe device on the GPU box, so the "SSD" is a file opened O_DIRECT (R19, section 13); what is compared
does not depend on the medium: the placement, the LBA range of every offload set (length = the paper's ceil formula), the
bytes of every sector of those ranges — read back from the file with plain Python file I/O, never through the library —
against orc_ssd_direct_store, every KV cache's GLT location against orc_ssd_location, and the retrieved paged tensors.
Bit-exact; nothing the library wrote is ever an expected value."""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import workloads as W

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(300)]

PATHS = {"staged": kv.PATH_STAGED, "zerocopy": kv.PATH_ZEROCOPY, "auto": kv.PATH_AUTO, "hybrid": kv.PATH_HYBRID}
KERNELS = {"vec16": kv.KERNEL_VEC16, "bulk": kv.KERNEL_BULK}
FILL = 0xC3                                      # what a stand-in file holds before anything is stored


@pytest.fixture(scope="module", autouse=True)
def _built():
    kvbuild.build()
    assert torch.cuda.is_available()
    kv.lib()


def _custom(geom, nphys, tables, n_dev, weights, cfg=78):
    return W.Workload(cfg, "custom", geom, (0,), nphys, [W.Request(np.asarray(t, dtype=np.int32)) for t in tables], n_dev, weights)


def _backing_file(path, nbytes):
    """A stand-in 'SSD' pre-filled with a pattern, so that sectors the library must not touch are recognisable."""
    with open(path, "wb") as f:
        f.write(bytes([FILL]) * nbytes)
    return str(path)


_LOOPS = []                                       # loop devices attached by _ssd_pool(blockdev=True), detached by _detach_loops


def _attach_loop(path):
    """A loop device over `path` (direct I/O to the backing file): a real block device node for the S_ISBLK branch."""
    import subprocess
    try:
        r = subprocess.run(["losetup", "-f", "--show", "--direct-io=on", str(path)], capture_output=True, text=True, timeout=30)
    except (OSError, subprocess.TimeoutExpired) as e:
        pytest.skip(f"no losetup here: {e}")
    if r.returncode != 0:
        pytest.skip(f"no loop device to be had here: {r.stderr.strip()}")
    _LOOPS.append(r.stdout.strip())
    return r.stdout.strip()


def _detach_loops():
    import subprocess
    while _LOOPS:
        subprocess.run(["losetup", "-d", _LOOPS.pop()], capture_output=True)


def _ssd_pool(wl, types, tmp_path, *, sector=512, slack=1.5, tuning=None, path=kv.PATH_AUTO, kernel=kv.KERNEL_VEC16, bandwidth=None, blockdev=False):
    """types[i] in {"mem", "ssd", "hbm"}; returns (pool, bw, files) with files[i] the backing file of SSD device i (with
    blockdev: the loop device attached to it, which is then what the pool opens)."""
    g = wl.geom
    bw = list(bandwidth) if bandwidth is not None else list(wl.default_weights())
    share = np.array(bw) / np.sum(bw)
    caps = [int(wl.moved_bytes() * s * slack) + (g.n_layers * len(wl.requests) + 4) * (g.payload + 2 * 65536) for s in share]
    caps = [(c + 65535) // 65536 * 65536 for c in caps]
    flags = [{"mem": 0, "ssd": kv.DEV_SSD, "hbm": kv.DEV_HBM}[t] for t in types]
    files = [_backing_file(tmp_path / f"ssd{i}.img", caps[i]) if t == "ssd" else None for i, t in enumerate(types)]
    if blockdev:
        files = [_attach_loop(f) if f else None for f in files]
    pool = kv.KvPool(bw, caps, n_layers=g.n_layers, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim, block_tokens=g.block_tokens,
                     elem_bytes=g.elem_bytes, dev_flags=flags, paths=files, sector_bytes=[sector if t == "ssd" else 0 for t in types])
    pool.set_path(path)
    pool.set_tuning(kernel=kernel, link_kernel=kernel, **(tuning or {}))
    return pool, bw, files


def _read_file(path, off, n):
    with open(path, "rb") as f:
        f.seek(off)
        return np.frombuffer(f.read(n), dtype=np.uint8)


def _check_ssd_stripe(pool, pl, l, i, path, want_stripe, payload, opl_l, seen_ranges):
    """Device i's LBA range of layer l against the oracle: length, sector bytes (payloads, zero padding), GLT locations."""
    first, n_sec, sec = pl.ssd_range(l, i)
    c = int(opl_l.counts[i])
    assert n_sec == oracle.lba_range_len(c, payload, sec) == kv.kvpool_plan_lba_range(c, payload, sec)
    assert pl.stripe_location(l, i) == (first, c * payload)
    for a, b in seen_ranges.setdefault(i, []):                          # ranges of one device never overlap
        assert first + n_sec <= a or b <= first
    seen_ranges[i].append((first, first + n_sec))
    info = pool.device_info(i)
    assert info["host_base"] in (None, 0) and (first + n_sec) * sec <= info["capacity"]
    disk = np.full((n_sec + 2) * sec, FILL, dtype=np.uint8)            # the oracle's disk: this range with a sector on either side
    assert oracle.ssd_direct_store(disk, sec, 1, want_stripe, payload) == n_sec
    lo = max(first - 1, 0)
    have = _read_file(path, lo * sec, (first - lo + n_sec + 1) * sec)
    assert np.array_equal(have[(first - lo) * sec:(first - lo + n_sec) * sec], disk[sec:(n_sec + 1) * sec]), f"sectors of layer {l} device {i} differ"
    assert np.array_equal(pl.stripe(l, i), want_stripe)                  # and through kvpool_stripe_read
    return first, n_sec, sec, have, lo


def _run(wl, types, tmp_path, *, path="auto", kernel="vec16", sector=512, tuning=None, bandwidth=None, batched=False, blockdev=False):
    dev = torch.device("cuda:0")
    g = wl.geom
    pool, bw, files = _ssd_pool(wl, types, tmp_path, sector=sector, tuning=tuning, path=PATHS[path], kernel=KERNELS[kernel], bandwidth=bandwidth,
                                blockdev=blockdev)
    try:
        for i, t in enumerate(types):
            assert pool.device_type(i)[0] == {"mem": kv.TYPE_MEM, "ssd": kv.TYPE_SSD, "hbm": kv.TYPE_HBM}[t]
        R, L = len(wl.requests), g.n_layers
        stream = torch.cuda.Stream()
        pls = [pool.place(wl.blocks_per_layer(r)) for r in range(R)]
        opls = [oracle.place(bw, wl.blocks_per_layer(r)) for r in range(R)]
        tables_np = [[np.ascontiguousarray(wl.layer_table(r, l)) for l in range(L)] for r in range(R)]
        tables = [[torch.from_numpy(t).to(dev) for t in row] for row in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for _ in range(L)]
        torch.cuda.synchronize()
        for r in range(R):
            for l in range(L):
                assert np.array_equal(pls[r].counts(l), opls[r][l].counts)
                d, s = pls[r].layer_map(l)
                assert np.array_equal(d.astype(np.uint32), opls[r][l].dev) and np.array_equal(s, opls[r][l].slot)
        for r in range(R):
            if batched:
                pool.offload_layers(pls[r], 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables[r], stream)
            else:
                for l in range(L):
                    pool.offload(pls[r], l, src[l][0], src[l][1], g.kvb, tables[r][l], stream)
        for r in range(R):
            pool.wait_offloads(pls[r], stream)
        stream.synchronize()                                               # wait_offloads: the store commands are on the disk by now
        seen = {}
        n_ssd_bytes = 0
        for r in range(R):
            for l in range(L):
                src_cpu = W.kv_layer_numpy(wl, l)
                want = oracle.offload_layer(src_cpu, tables_np[r][l], opls[r][l])
                for i, t in enumerate(types):
                    if t != "ssd":
                        assert np.array_equal(pls[r].stripe(l, i), want[i]), (r, l, i)
                        continue
                    first, n_sec, sec, _, _ = _check_ssd_stripe(pool, pls[r], l, i, files[i], want[i], g.payload, opls[r][l], seen)
                    n_ssd_bytes += want[i].nbytes
                K = len(tables_np[r][l])
                for j in ([0, K - 1] + list(np.random.default_rng(l).integers(0, K, size=min(K, 24)))) if K else []:
                    d, ty, s, loc = pls[r].lookup(l, int(j))
                    assert (d, s) == (int(opls[r][l].dev[j]), int(opls[r][l].slot[j]))
                    if types[d] != "ssd":
                        continue
                    first, _, sec = pls[r].ssd_range(l, d)
                    lba, off = pls[r].ssd_location(l, int(j))
                    assert (lba, off) == oracle.ssd_location(first, s, g.payload, sec) and ty == kv.TYPE_SSD and loc == lba
                    got = _read_file(files[d], lba * sec + off, g.payload)   # SSD_Direct_Retrieve of one KV cache, by hand
                    assert np.array_equal(got, want[d][s * g.payload:(s + 1) * g.payload])
        for r in range(R):
            if batched:
                pool.retrieve_layers(pls[r], 0, [x[0] for x in dst], [x[1] for x in dst], g.kvb, tables[r], stream)
            else:
                for l in range(L):
                    pool.retrieve(pls[r], l, dst[l][0], dst[l][1], g.kvb, tables[r][l], stream)
        stream.synchronize()
        pool.synchronize()
        for l in range(L):
            src_cpu = W.kv_layer_numpy(wl, l)
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            for r in range(R):
                want = oracle.offload_layer(src_cpu, tables_np[r][l], opls[r][l])
                oracle.retrieve_layer(ref, tables_np[r][l], opls[r][l], want)
            assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), ref), f"retrieved layer {l} differs from the oracle"
        infos = {i: pool.ssd_info(i) for i, t in enumerate(types) if t == "ssd"}
        for pl in pls:
            pl.release()
        assert all(pool.device_info(i)["used"] == 0 for i in range(pool.n_devices))
        return {"ssd_bytes": n_ssd_bytes, "info": infos}
    finally:
        pool.destroy()
        _detach_loops()


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["auto", "staged", "zerocopy", "hybrid"])
def test_host_memory_plus_ssd_pool_llama_1k(tmp_path, path, kernel):
    """Config 1's shape (LLaMA-3.1-8B at 1K, 4 layers) over the paper's own mix: one host-memory device and one SSD, 2:1."""
    wl = W.make_workload(1, n_layers=4)
    out = _run(wl, ["mem", "ssd"], tmp_path, path=path, kernel=kernel)
    assert out["ssd_bytes"] == 4 * 21 * wl.geom.payload              # device 1 holds 21 of the 64 blocks of every layer
    info = out["info"][1]
    assert info["sector_bytes"] == 512 and not info["block_device"] and info["stores"] >= 4 and info["retrieves"] >= 4
    assert info["queue_depth"] in (1, 8)                             # io_uring with 2 x 4 lanes in flight, or the synchronous fall-back


@pytest.mark.parametrize("sector", [512, 4096])
def test_ssd_only_pool_and_two_ssds(tmp_path, sector):
    wl = W.make_workload(1, n_layers=3)
    wl1 = _custom(wl.geom, wl.nphys, [wl.requests[0].table], 1, (1.0,))
    _run(wl1, ["ssd"], tmp_path, sector=sector)
    (tmp_path / "b").mkdir()
    _run(wl, ["ssd", "ssd"], tmp_path / "b", sector=sector, batched=True)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_commands_smaller_than_a_stripe_and_every_device_type_in_one_pool(tmp_path, kernel):
    """Config 4's shape at 1/16 (512 blocks of 32 KiB per layer) over host memory, two SSDs and an HBM-type device, with 1 MiB
    commands on 2 lanes: a stripe travels in several commands and the lanes are recycled many times."""
    wl = W.make_workload(4, scale=1 / 16, n_layers=3)
    wl = _custom(wl.geom, wl.nphys, [wl.requests[0].table], 4, (4.0, 2.0, 1.0, 4.0), cfg=4)
    out = _run(wl, ["mem", "ssd", "ssd", "hbm"], tmp_path, kernel=kernel, tuning={"ssd_lanes": 2, "ssd_chunk_bytes": 1 << 20}, batched=True)
    # device 1: 2/11 of 512 blocks = 93 or 94 blocks of 32 KiB per layer ~ 2.9 MiB: at least 3 commands per layer and direction
    assert out["info"][1]["stores"] >= 9 and out["info"][1]["retrieves"] >= 9


@pytest.mark.parametrize("sector", [512, 4096])
def test_kv_size_that_is_not_a_multiple_of_the_sector(tmp_path, sector):
    """PAPER.md:183's ceiling matters when KV_size is not a sector multiple: P = 2 * 16 * 1 * 80 * 2 = 5120 B (ten 512-byte
    sectors, 1.25 sectors of 4 KiB) and P = 96 B; ranges end inside a sector (zero padding), commands start inside one."""
    rng = np.random.default_rng(6)
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=80)
    _run(_custom(g, 301, [rng.permutation(301)[:257]], 3, (3.0, 2.0, 1.0)), ["mem", "ssd", "ssd"], tmp_path, sector=sector,
         tuning={"ssd_lanes": 2, "ssd_chunk_bytes": 64 << 10})
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=24, block_tokens=1)       # kvb = 48, P = 96
    (tmp_path / "b").mkdir()
    _run(_custom(g, 900, [rng.permutation(900)[:777]], 2, (1.0, 2.0)), ["mem", "ssd"], tmp_path / "b", sector=sector,
         tuning={"ssd_lanes": 3, "ssd_chunk_bytes": 4096})
    # K < N: a device that receives nothing has an empty range
    g = W.Geometry(n_layers=1, n_kv_heads=2, head_dim=64)
    (tmp_path / "c").mkdir()
    _run(_custom(g, 9, [[7, 2]], 3, (4.0, 2.0, 1.0)), ["mem", "ssd", "ssd"], tmp_path / "c", sector=sector)


@pytest.mark.parametrize("sector", [512, 4096])
def test_instalments_and_partial_retrieval_on_an_ssd(tmp_path, sector):
    """kvpool_offload_range / kvpool_retrieve_range with an SSD in the pool: instalments that start and
    end inside a sector (P = 1536 B) must keep their neighbours' bytes (read-modify-write of the edge sectors); every
    intermediate state of the LBA ranges equals the oracle's stripes stored by orc_ssd_direct_store."""
    rng = np.random.default_rng(8)
    g = W.Geometry(n_layers=1, n_kv_heads=3, head_dim=16, block_tokens=8)       # kvb = 768, P = 1536
    wl = _custom(g, 400, [rng.permutation(400)[:333]], 2, (1.0, 1.0))
    dev = torch.device("cuda:0")
    pool, bw, files = _ssd_pool(wl, ["ssd", "mem"], tmp_path, sector=sector, tuning={"ssd_lanes": 2, "ssd_chunk_bytes": 32 << 10})
    try:
        pl = pool.place(wl.blocks_per_layer(0))
        opl = oracle.place(bw, wl.blocks_per_layer(0))[0]
        table_np = np.ascontiguousarray(wl.layer_table(0, 0))
        K = len(table_np)
        table = torch.from_numpy(table_np).to(dev)
        src, src_cpu = W.kv_layer_torch(wl, 0, dev), W.kv_layer_numpy(wl, 0)
        first, n_sec, sec = pl.ssd_range(0, 0)
        stripes = [np.full(int(c) * g.payload, FILL, dtype=np.uint8) for c in opl.counts]
        cuts = [0, 5, 6, 100, 101, 250, K]
        order = [2, 0, 4, 1, 5, 3]                                           # instalments arrive out of order
        done = np.zeros(K, bool)
        for step, q in enumerate(order):
            a, b = cuts[q], cuts[q + 1]
            if step == 2:                                                      # a block that has not arrived yet: ESTATE
                with pytest.raises(kv.KvPoolError) as e:
                    pool.retrieve_range(pl, 0, cuts[1], 1, src[0], src[1], g.kvb, table)
                assert e.value.code == kv.ESTATE
            pool.offload_range(pl, 0, a, b - a, src[0], src[1], g.kvb, table)
            oracle.offload_range(src_cpu, table_np, opl, stripes, a, b - a)
            done[a:b] = True
            pool.wait_offloads(pl)
            torch.cuda.synchronize()
            # the slots stored so far equal the oracle's; the file outside the range is untouched
            have = _read_file(files[0], first * sec, n_sec * sec)
            slots = np.array([int(opl.slot[j]) for j in range(K) if opl.dev[j] == 0 and done[j]], dtype=np.int64)
            got = have[:int(opl.counts[0]) * g.payload].reshape(-1, g.payload)
            assert np.array_equal(got[slots], stripes[0].reshape(-1, g.payload)[slots]), f"after instalment {step}"
            assert (_read_file(files[0], (first + n_sec) * sec, sec) == FILL).all()
            if first:
                assert (_read_file(files[0], (first - 1) * sec, sec) == FILL).all()
        # complete: the whole range equals SSD_Direct_Store of the full stripe, zero padding included
        disk = np.full(n_sec * sec, FILL, dtype=np.uint8)
        assert oracle.ssd_direct_store(disk, sec, 0, stripes[0], g.payload) == n_sec
        assert np.array_equal(_read_file(files[0], first * sec, n_sec * sec), disk)
        for a, n in [(0, K), (0, 1), (K - 1, 1), (3, 0), (17, 90), (200, 133), (5, 1)]:
            dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
            pool.retrieve_range(pl, 0, a, n, dst[0], dst[1], g.kvb, table)
            torch.cuda.synchronize()
            want = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_range(want, table_np, opl, stripes, a, n)
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), want), (a, n)
        pl.release()
    finally:
        pool.destroy()


def test_lba_ranges_are_recycled_and_several_requests_share_a_device(tmp_path):
    """Two live placements on one SSD hold disjoint ranges; a released placement's range is handed out again; a re-offload of
    the same layer replaces its sectors; a retrieve enqueued straight after an offload (no wait) reads the new bytes."""
    wl = W.make_workload(1, n_layers=2)
    g, dev = wl.geom, torch.device("cuda:0")
    pool, bw, files = _ssd_pool(wl, ["mem", "ssd"], tmp_path, slack=3.0)
    try:
        bpl = wl.blocks_per_layer(0)
        opl = oracle.place(bw, bpl)
        table_np = np.ascontiguousarray(wl.layer_table(0, 0))
        table = torch.from_numpy(table_np).to(dev)
        a, b = pool.place(bpl), pool.place(bpl)
        ra, rb = [a.ssd_range(l, 1) for l in range(2)], [b.ssd_range(l, 1) for l in range(2)]
        spans = sorted((f, f + n) for f, n, _ in ra + rb)
        assert all(x[1] <= y[0] for x, y in zip(spans, spans[1:]))
        a.release()
        c = pool.place(bpl)
        assert [c.ssd_range(l, 1) for l in range(2)] == ra                    # first fit: the freed range again
        for gen in range(2):                                                   # second pass: other bytes into the same sectors
            wl2 = W.make_workload(1, n_layers=2) if gen == 0 else _custom(g, wl.nphys, [wl.requests[0].table], 2, (2.0, 1.0), cfg=31)
            src, src_cpu = W.kv_layer_torch(wl2, 0, dev), W.kv_layer_numpy(wl2, 0)
            dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
            pool.offload(c, 0, src[0], src[1], g.kvb, table)
            pool.retrieve(c, 0, dst[0], dst[1], g.kvb, table)                 # no wait in between: the worker keeps the order
            torch.cuda.synchronize()
            pool.synchronize()
            want = oracle.offload_layer(src_cpu, table_np, opl[0])
            first, n_sec, sec = c.ssd_range(0, 1)
            disk = np.zeros(n_sec * sec, dtype=np.uint8)
            oracle.ssd_direct_store(disk, sec, 0, want[1], g.payload)
            assert np.array_equal(_read_file(files[1], first * sec, n_sec * sec), disk)
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, table_np, opl[0], want)
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref)
        b.release()
        c.release()
    finally:
        pool.destroy()


def test_ssd_errors_bad_arguments_full_device_and_a_failing_disk(tmp_path):
    g = W.Geometry(n_layers=1, n_kv_heads=8, head_dim=128)
    geo = dict(n_layers=1, n_kv_heads=8, head_dim=128)
    with pytest.raises(kv.KvPoolError) as e:                                   # an SSD without a path
        kv.KvPool([1.0], [1 << 20], dev_flags=[kv.DEV_SSD], **geo)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                   # a path on a host-memory device
        kv.KvPool([1.0], [1 << 20], paths=[str(tmp_path / "x")], **geo)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                   # SSD excludes the other flags
        kv.KvPool([1.0], [1 << 20], dev_flags=[kv.DEV_SSD | kv.DEV_HBM], paths=[str(tmp_path / "x")], **geo)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                   # two devices on one path: their LBA ranges would overlap
        kv.KvPool([1.0, 1.0], [1 << 20] * 2, dev_flags=[kv.DEV_SSD] * 2, paths=[str(tmp_path / "x")] * 2, **geo)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                   # sector size not a power of two
        kv.KvPool([1.0], [1 << 20], dev_flags=[kv.DEV_SSD], paths=[str(tmp_path / "x")], sector_bytes=[520], **geo)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                   # a directory that does not exist
        kv.KvPool([1.0], [1 << 20], dev_flags=[kv.DEV_SSD], paths=[str(tmp_path / "no" / "such" / "dir" / "x")], **geo)
    assert e.value.code == kv.EIO
    assert not (tmp_path / "x").exists()                                       # failed creates leave nothing behind

    # a file the library creates itself goes away with the pool; a full device refuses a placement and reserves nothing
    path = tmp_path / "made.img"
    pool = kv.KvPool([1.0], [4 * g.payload + 4096], dev_flags=[kv.DEV_SSD], paths=[str(path)], sector_bytes=[512], **geo)
    assert path.exists() and pool.device_type(0) == (kv.TYPE_SSD, -1)
    with pytest.raises(kv.KvPoolError) as e:
        pool.place([5])
    assert e.value.code == kv.ENOMEM and pool.device_info(0)["used"] == 0
    pl = pool.place([4])
    with pytest.raises(kv.KvPoolError) as e:                                   # lanes exist now: their size is fixed
        pool.set_tuning(ssd_lanes=8)
    assert e.value.code == kv.ESTATE
    with pytest.raises(kv.KvPoolError) as e:
        pl.ssd_location(0, 4)
    assert e.value.code == kv.EINVAL
    pl.release()
    pool.destroy()
    assert not path.exists()

    # a disk that fails under the pool: the commands complete their handshakes (nothing hangs) and the failure surfaces as EIO
    wl = W.make_workload(1, n_layers=1)
    dev = torch.device("cuda:0")
    pool, bw, files = _ssd_pool(wl, ["ssd"], tmp_path, bandwidth=[1.0])
    wl = _custom(wl.geom, wl.nphys, [wl.requests[0].table], 1, (1.0,))
    try:
        pl = pool.place(wl.blocks_per_layer(0))
        table = torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, 0))).to(dev)
        src = W.kv_layer_torch(wl, 0, dev)
        pool.offload(pl, 0, src[0], src[1], wl.geom.kvb, table)
        pool.wait_offloads(pl)
        torch.cuda.synchronize()
        pool.synchronize()
        assert pool.io_errors() == 0
        # leave recognisable bytes in the retrieve lanes: a retrieve that works, of KV that is all 0x77
        marker = torch.full((2, wl.nphys, wl.geom.kvb), 0x77, dtype=torch.uint8, device=dev)
        pool.offload(pl, 0, marker[0], marker[1], wl.geom.kvb, table)
        pool.wait_offloads(pl)
        pool.retrieve(pl, 0, marker[0], marker[1], wl.geom.kvb, table)
        pool.offload(pl, 0, src[0], src[1], wl.geom.kvb, table)
        pool.wait_offloads(pl)
        torch.cuda.synchronize()
        pool.synchronize()
        assert pool.io_errors() == 0
        os.truncate(files[0], 0)                                               # the device loses its sectors
        dst = W.poison_torch((2, wl.nphys, wl.geom.kvb // 2), dev)
        pool.retrieve(pl, 0, dst[0], dst[1], wl.geom.kvb, table)
        torch.cuda.synchronize()                                               # returns: the failed reads still release their lanes
        assert pool.io_errors() > 0                                            # visible without blocking, before any synchronize
        # what the failed commands handed over is zero bytes: neither the lanes' last contents (0x77) nor anything else
        got = dst.view(torch.uint8).reshape(2, wl.nphys, wl.geom.kvb)[:, table.long()]
        assert int(got.count_nonzero()) == 0
        with pytest.raises(kv.KvPoolError) as e:
            pool.synchronize()
        assert e.value.code == kv.EIO
        pool.synchronize()                                                     # reported once
        pl.release()
    finally:
        pool.destroy()


def test_wait_offloads_covers_every_command_of_a_stripe_and_every_instalment(tmp_path):
    """A stripe much larger than a lane is many store commands spread over the lanes, an instalment offload adds more, and
    the worker completes them in whatever order the disk does: after kvpool_wait_offloads + a sync of THAT stream (no
    kvpool_synchronize, no stripe read through the library, both of which would wait for the worker) every sector of the
    stripe must already be in the file."""
    base = W.make_workload(1, n_layers=8)                                       # 64 KV caches of 64 KiB per layer
    wl = _custom(base.geom, base.nphys, [base.requests[0].table], 1, (1.0,))
    g = wl.geom
    dev = torch.device("cuda:0")
    pool, bw, files = _ssd_pool(wl, ["ssd"], tmp_path, bandwidth=[1.0], tuning={"ssd_chunk_bytes": 3 * g.payload, "ssd_lanes": 4})
    try:
        bpl = wl.blocks_per_layer(0)
        pl = pool.place(bpl)
        opl = oracle.place(bw, bpl)
        stream = torch.cuda.Stream()
        srcs = [W.kv_layer_torch(wl, l, dev) for l in range(g.n_layers)]
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(g.n_layers)]
        tables = [torch.from_numpy(t).to(dev) for t in tables_np]
        torch.cuda.synchronize()
        for l in range(g.n_layers):
            K = int(bpl[l])
            cuts = [0, K] if l % 2 == 0 else [0, K // 3, K // 3 + 5, K]           # odd layers arrive in three instalments
            for a, b in zip(cuts, cuts[1:]):
                pool.offload_range(pl, l, a, b - a, srcs[l][0], srcs[l][1], g.kvb, tables[l], stream)
            pool.wait_offloads(pl, stream)
            stream.synchronize()
            first, n_sec, sec = pl.ssd_range(l, 0)
            want = oracle.offload_layer(W.kv_layer_numpy(wl, l), tables_np[l], opl[l])[0]
            have = _read_file(files[0], first * sec, want.nbytes)
            assert np.array_equal(have, want), f"layer {l}: wait_offloads returned before every store command was on the disk"
        assert pool.ssd_info(0)["stores"] >= g.n_layers * 20                      # really many commands per stripe
        pool.synchronize()
        pl.release()
    finally:
        pool.destroy()


def test_measure_bandwidth_and_calibrate_with_an_ssd(tmp_path):
    """kvpool_measure_bandwidth on an SSD-type device times the device's own sequential commands; kvpool_calibrate feeds the
    result to Eq. 1, and the placement that follows equals the oracle's for those bandwidths."""
    wl = W.make_workload(1, n_layers=1)
    pool, _, files = _ssd_pool(wl, ["mem", "ssd"], tmp_path, slack=40.0)
    try:
        r = pool.measure_bandwidth(1, kv.MEASURE_RETRIEVE, 32 << 20, 3)
        w = pool.measure_bandwidth(1, kv.MEASURE_OFFLOAD, 32 << 20, 3)
        assert 0.01 < r < 1000 and 0.01 < w < 1000
        b = pool.calibrate(kv.MEASURE_RETRIEVE, 32 << 20, 3)
        assert np.array_equal(pool.weights(), oracle.weights(b))
        pl = pool.place(wl.blocks_per_layer(0))
        opl = oracle.place(list(b), wl.blocks_per_layer(0))
        assert np.array_equal(pl.counts(0), opl[0].counts)
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.timeout(1200)
def test_full_size_config4_with_two_ssd_devices_every_byte_against_oracle(tmp_path):
    """BASELINE.json's headline configuration at its FULL size (Qwen3-30B-A3B-shaped KV at 128K: 48 layers x 8192 blocks, 12 GiB
    per leg, weights 4:4:2:2:1:1) with the two slowest pool devices made SSD-type: 585 blocks of every layer (18.3 MiB, three
    8 MiB commands) go to each, 1.7 GiB in all through the lanes.  Batched calls as in bench.py; compared with the oracle
    BYTE FOR BYTE, streamed layer by layer: every stripe, every sector of every LBA range (read from the files with plain file
    I/O), the whole retrieved tensor."""
    wl = W.make_workload(4)
    g, dev, L = wl.geom, torch.device("cuda:0"), wl.geom.n_layers
    bw = list(wl.default_weights())
    types = ["mem"] * 4 + ["ssd"] * 2
    share = np.array(bw) / np.sum(bw)
    caps = [(int(wl.moved_bytes() * s * 1.1) + (L + 4) * (g.payload + 8192) + 65535) // 65536 * 65536 for s in share]
    files = [str(tmp_path / f"ssd{i}.img") if t == "ssd" else None for i, t in enumerate(types)]
    pool = kv.KvPool(bw, caps, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim, dev_flags=[kv.DEV_SSD if t == "ssd" else 0 for t in types],
                     paths=files, sector_bytes=[4096 if t == "ssd" else 0 for t in types], link_groups=[1] * 6)
    try:
        bpl = wl.blocks_per_layer(0)
        pl, opl = pool.place(bpl), oracle.place(bw, bpl)
        table_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) for t in table_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for _ in range(L)]
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, s)
        pool.wait_offloads(pl, s)
        s.synchronize()
        pool.synchronize()
        pool.retrieve_layers(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, s)
        s.synchronize()
        pool.synchronize()
        shape = (2, wl.nphys, g.kvb // 2)
        pin_src, pin_got = torch.empty(shape, dtype=torch.int16).pin_memory(), torch.empty(shape, dtype=torch.int16).pin_memory()
        ref = np.empty(shape, dtype=np.uint16)
        stripe_bytes = sector_bytes = 0
        for l in range(L):
            assert np.array_equal(pl.counts(l), opl[l].counts) and list(opl[l].counts) == [2341, 2341, 1170, 1170, 585, 585]
            d_, s_ = pl.layer_map(l)
            assert np.array_equal(d_.astype(np.uint32), opl[l].dev) and np.array_equal(s_, opl[l].slot)
            pin_src.copy_(src[l], non_blocking=True)
            pin_got.copy_(dst[l], non_blocking=True)
            torch.cuda.synchronize()
            src_cpu, got = pin_src.numpy().view(np.uint16), pin_got.numpy().view(np.uint16)
            want = oracle.offload_layer(src_cpu, table_np[l], opl[l], parallel=True)
            for i, t in enumerate(types):
                assert np.array_equal(pl.stripe(l, i), want[i]), f"stripe bytes differ: layer {l} device {i}"
                stripe_bytes += want[i].nbytes
                if t == "ssd":
                    first, n_sec, sec = pl.ssd_range(l, i)
                    assert n_sec == oracle.lba_range_len(585, g.payload, sec) == 585 * 8
                    disk = np.empty(n_sec * sec, dtype=np.uint8)
                    oracle.ssd_direct_store(disk, sec, 0, want[i], g.payload)
                    assert np.array_equal(_read_file(files[i], first * sec, n_sec * sec), disk), f"sectors differ: layer {l} device {i}"
                    sector_bytes += disk.nbytes
            ref[...] = W.POISON_BITS
            oracle.retrieve_layer(ref, table_np[l], opl[l], want, parallel=True)
            assert np.array_equal(got, ref), f"retrieved layer {l} differs from the oracle's"
        assert stripe_bytes == wl.moved_bytes() and sector_bytes == 2 * 48 * 585 * g.payload
        info = pool.ssd_info(5)
        assert info["stores"] >= 48 * 3 and info["retrieves"] >= 48 * 3
        pl.release()
    finally:
        pool.destroy()


def test_synchronous_fallback_of_the_worker(tmp_path, monkeypatch):
    """KVPOOL_SSD_SYNC=1 (or a kernel without io_uring): one pread / pwrite at a time instead of a ring of commands in flight;
    same bytes."""
    monkeypatch.setenv("KVPOOL_SSD_SYNC", "1")
    wl = W.make_workload(1, n_layers=2)
    out = _run(wl, ["mem", "ssd"], tmp_path, tuning={"ssd_lanes": 2, "ssd_chunk_bytes": 256 << 10})
    assert out["info"][1]["queue_depth"] == 1


@pytest.mark.timeout(180)
def test_ssd_pool_makes_progress_next_to_another_pools_copy_engine_traffic(tmp_path):
    """Two pools on two host threads: one streams a host-memory pool's 128 MiB layers through the copy engines without a
    pause, the other offloads and retrieves through an SSD-type device.  The SSD pool's lanes use no copy engine and their
    stream wait-values sit on compute streams, so they neither starve nor stall the other pool (a first version that staged
    lanes through cudaMemcpyAsync stopped making progress in exactly this set-up: kvpool_ssd.cu).  Results against the
    oracle; the whole test must finish in seconds."""
    import threading
    import time
    wl = W.make_workload(2, scale=1 / 4, n_layers=4)                     # LLaMA-shaped, 512 blocks of 64 KiB per layer = 32 MiB
    g, dev, L = wl.geom, torch.device("cuda:0"), 4
    big = W.make_workload(2, n_layers=2)                                 # the other pool's request: 2 layers of 128 MiB
    bpl_big = big.blocks_per_layer(0)
    mem = kv.KvPool([1.0], [big.moved_bytes() + (1 << 20)], n_layers=2, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim)
    pool, bw, files = _ssd_pool(_custom(g, wl.nphys, [wl.requests[0].table], 1, (1.0,), cfg=2), ["ssd"], tmp_path, sector=4096)
    stop, rounds, errors = threading.Event(), [0], []
    try:
        big_src = [W.kv_layer_torch(big, l, dev) for l in range(2)]
        big_tab = [torch.from_numpy(np.ascontiguousarray(big.layer_table(0, l))).to(dev) for l in range(2)]
        plm = mem.place(bpl_big)
        s2 = torch.cuda.Stream()
        mem.offload_layers(plm, 0, [x[0] for x in big_src], [x[1] for x in big_src], g.kvb, big_tab, s2)
        mem.wait_offloads(plm, s2)
        s2.synchronize()

        def background():
            try:
                while not stop.is_set():
                    mem.offload_layers(plm, 0, [x[0] for x in big_src], [x[1] for x in big_src], g.kvb, big_tab, s2)
                    mem.retrieve_layers(plm, 0, [x[0] for x in big_src], [x[1] for x in big_src], g.kvb, big_tab, s2)   # (a round trip onto itself)
                    s2.synchronize()
                    rounds[0] += 1
            except Exception as e:                                         # pragma: no cover
                errors.append(e)

        th = threading.Thread(target=background)
        th.start()
        time.sleep(0.05)
        t0 = time.perf_counter()
        bpl = wl.blocks_per_layer(0)
        pl, opl = pool.place(bpl), oracle.place([1.0], bpl)
        s1 = torch.cuda.Stream()
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) for t in tables_np]
        for rep in range(3):
            src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
            dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for _ in range(L)]
            torch.cuda.current_stream().synchronize()
            pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, s1)
            pool.retrieve_layers(pl, 0, [x[0] for x in dst], [x[1] for x in dst], g.kvb, tables, s1)
            s1.synchronize()
            for l in range(L):
                want = oracle.offload_layer(W.kv_layer_numpy(wl, l), tables_np[l], opl[l])
                ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
                oracle.retrieve_layer(ref, tables_np[l], opl[l], want)
                assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), ref), (rep, l)
        took = time.perf_counter() - t0
        stop.set()
        th.join(60)
        assert not th.is_alive() and not errors, errors
        assert rounds[0] >= 2                                              # the other pool kept streaming meanwhile
        assert took < 60, took                                             # 768 MiB through the "disk" and back: seconds, not a stall
        pool.synchronize()
        pl.release()
        plm.release()
    finally:
        stop.set()
        pool.destroy()
        mem.destroy()


def test_per_layer_events_with_an_ssd_in_the_pool(tmp_path):
    """kvpool_retrieve_layers_signal over host memory + an SSD-type device (layerwise pipelining): a layer's
    event fires once the host buffer's share AND the SSD's share of that layer are in the paged layout; a consumer that waits
    on nothing but the events reads the oracle's bytes."""
    wl = W.make_workload(1, n_layers=6)
    g, dev, L = wl.geom, torch.device("cuda:0"), 6
    pool, bw, files = _ssd_pool(wl, ["mem", "ssd"], tmp_path, tuning={"ssd_lanes": 2, "ssd_chunk_bytes": 512 << 10})
    try:
        bpl = wl.blocks_per_layer(0)
        pl = pool.place(bpl)
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) for t in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for _ in range(L)]
        sums = torch.zeros(L, dtype=torch.int64, device=dev)
        torch.cuda.synchronize()
        io, consumer = torch.cuda.Stream(), torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, io)
        ready = [torch.cuda.Event() for _ in range(L)]
        pool.retrieve_layers_signal(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, ready, io)   # (no wait in between)
        pool.checksum_layers([d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, bpl, ready, sums, consumer)
        consumer.synchronize()
        got = [int(x) % 2 ** 64 for x in sums.cpu().tolist()]
        assert got == [oracle.checksum(W.kv_layer_numpy(wl, l), tables_np[l]) for l in range(L)]
        io.synchronize()
        for l in range(L):
            assert torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()])
        pool.synchronize()
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("sector", [0, 4096])
def test_ssd_type_device_on_a_block_device_node(tmp_path, sector):
    """The S_ISBLK branch (no NVMe on the box: a loop device, itself doing direct I/O to its backing file, is the block device
    node): capacity checked against BLKGETSIZE64, the sector size taken from BLKSSZGET when the caller gives none, no file
    system between the library and the device's sectors — which are read back here through the device node, never through
    the library, and compared with orc_ssd_direct_store."""
    wl = W.make_workload(1, n_layers=3)
    out = _run(wl, ["mem", "ssd"], tmp_path, sector=sector, blockdev=True, batched=True, tuning={"ssd_lanes": 3, "ssd_chunk_bytes": 512 << 10})
    info = out["info"][1]
    assert info["block_device"] and info["sector_bytes"] == (sector or 512) and info["stores"] >= 3
    # a capacity beyond the device is refused
    f = _backing_file(tmp_path / "small.img", 1 << 20)
    loop = _attach_loop(f)
    try:
        with pytest.raises(kv.KvPoolError) as e:
            kv.KvPool([1.0], [2 << 20], dev_flags=[kv.DEV_SSD], paths=[loop], n_layers=1, n_kv_heads=8, head_dim=128)
        assert e.value.code == kv.EINVAL
    finally:
        _detach_loops()
    assert os.path.exists(f)                                                   # the library never removes what it did not create
