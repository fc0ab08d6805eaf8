"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol the header
declares, the pure-host placement entry points agree bit-for-bit with the oracle, and argument errors come back
as codes.  No kernel runs here."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA_LIB = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "lib64")


@pytest.fixture(scope="module", autouse=True)
def _built():
    kvbuild.build()


def test_library_exports_every_symbol_declared_in_header():
    pat = r"KVPOOL_API\s+(?:const\s+char\*|int)\s+(kvpool_\w+)\s*\("
    product = set(re.findall(pat, open(os.path.join(ROOT, "include", "kvpool.h")).read()))
    devel = set(re.findall(pat, open(os.path.join(ROOT, "include", "kvpool_dev.h")).read()))
    # the product header is the boundary SURVEY.md 8(b) lists; baselines, stand-ins, counters and profiling live apart
    assert devel == {"kvpool_offload_naive", "kvpool_retrieve_naive", "kvpool_checksum", "kvpool_checksum_layers", "kvpool_spin", "kvpool_stats",
                     "kvpool_set_profiling", "kvpool_profile_read", "kvpool_profile_read_clock"} and not (devel & product)
    declared = sorted(product | devel)
    assert len(declared) >= 27 and "kvpool_create" in declared and "kvpool_retrieve" in declared
    lib = ctypes.CDLL(kv.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"
    assert sorted(kv.EXPORTS) == declared                      # the Python binding mirrors the header one to one
    assert kv.version().startswith("kvpool")


def _cases(seed, n_cases, max_n=8, max_k=3000, max_w=60000):
    rng = np.random.default_rng(seed)
    for _ in range(n_cases):
        n = int(rng.integers(1, max_n + 1))
        w = rng.integers(1, max_w + 1, size=n)
        if rng.random() < 0.3:
            w[rng.integers(0, n, size=n // 2 + 1)] = w[0]
        yield [int(x) for x in w], int(rng.integers(0, max_k + 1))


def test_plan_layer_matches_oracle_bit_for_bit():
    for w, K in _cases(21, 1500):
        c, dev, slot = kv.kvpool_plan_layer(w, K)
        oc = oracle.counts(w, K)
        od, os_ = oracle.wrr(oc, K)
        assert np.array_equal(c, oc)
        assert np.array_equal(dev.astype(np.uint32), od) and np.array_equal(slot, os_)
    # many devices, large K, extreme weight ratios
    for w, K in _cases(22, 40, max_n=32, max_k=40000, max_w=10 ** 9):
        c, dev, slot = kv.kvpool_plan_layer(w, K)
        oc = oracle.counts(w, K)
        od, os_ = oracle.wrr(oc, K)
        assert np.array_equal(c, oc) and np.array_equal(dev.astype(np.uint32), od) and np.array_equal(slot, os_)


def test_plan_matches_oracle_on_all_baseline_configs():
    for cfg in (1, 2, 3, 4, 5, 6):
        wl = W.make_workload(cfg)
        bw = wl.default_weights()
        w = kv.kvpool_plan_weights(bw)
        assert np.array_equal(w, oracle.weights(bw))
        for r in range(len(wl.requests)):
            for K in sorted(set(int(k) for k in wl.blocks_per_layer(r))):
                c, dev, slot = kv.kvpool_plan_layer(w, K)
                oc = oracle.counts(w, K)
                od, os_ = oracle.wrr(oc, K)
                assert np.array_equal(c, oc) and np.array_equal(dev.astype(np.uint32), od) and np.array_equal(slot, os_)
    c = kv.kvpool_plan_layer(kv.kvpool_plan_weights((4, 4, 2, 2, 1, 1)), 8192, with_map=False)
    assert list(c) == [2341, 2341, 1170, 1170, 585, 585]


def test_plan_weights_quantisation_and_errors():
    b = [55.62, 57.26, 21.3, 0.001, 12.3456]
    assert np.array_equal(kv.kvpool_plan_weights(b), oracle.weights(b))
    for bad in ([1.0, 0.0], [-1.0], [0.0004], [float("nan")], [float("inf")], []):
        with pytest.raises(kv.KvPoolError) as e:
            kv.kvpool_plan_weights(bad)
        assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError):
        kv.kvpool_plan_weights([1.0] * 33)                     # more than KVPOOL_MAX_DEVICES
    with pytest.raises(kv.KvPoolError):
        kv.kvpool_plan_layer([1, 0, 1], 5)                     # zero weight


def test_share_bandwidth_divides_what_a_link_group_shares():
    """kvpool_share_bandwidth (include/kvpool.h): host arithmetic in front of Eq. 1, not part of the paper's method — checked
    against exact rational arithmetic: ungrouped devices keep their bandwidth, a group's shares add up to its best member's
    rate and keep the members' proportions, m equal members get 1/m each."""
    from fractions import Fraction
    rng = np.random.default_rng(5)
    for _ in range(200):
        n = int(rng.integers(1, 9))
        alone = [float(rng.integers(1, 4000)) / 8.0 for _ in range(n)]          # exactly representable
        groups = [int(x) for x in rng.integers(0, 4, size=n)]
        out = kv.kvpool_share_bandwidth(alone, groups)
        for g in set(groups):
            members = [i for i in range(n) if groups[i] == g]
            if g == 0:
                assert all(out[i] == alone[i] for i in members)
                continue
            best, total = max(Fraction(alone[i]) for i in members), sum(Fraction(alone[i]) for i in members)
            for i in members:
                exact = Fraction(alone[i]) * best / total
                assert abs(Fraction(float(out[i])) - exact) <= exact * Fraction(1, 2 ** 50)
                assert out[i] == alone[i] * float(best) / float(total)               # the header's left-to-right double formula
            assert abs(sum(Fraction(float(out[i])) for i in members) - best) <= best * Fraction(1, 2 ** 48)
    assert list(kv.kvpool_share_bandwidth([56.0, 56.0, 3000.0, 3000.0], [1, 1, 2, 2])) == [28.0, 28.0, 1500.0, 1500.0]
    assert list(kv.kvpool_share_bandwidth([56.0, 3000.0], [0, 0])) == [56.0, 3000.0]
    for bad in ([1.0, 0.0], [float("nan")], [float("inf")]):
        with pytest.raises(kv.KvPoolError) as e:
            kv.kvpool_share_bandwidth(bad, [1] * len(bad))
        assert e.value.code == kv.EINVAL


def test_validate_table_accepts_every_workload_table_and_names_the_offending_entry():
    """DESIGN.md R12: distinct entries in [0, nphys) are the caller's contract; the host-side checker states it."""
    for cfg in (1, 3, 5):
        wl = W.make_workload(cfg, scale=1 / 8) if cfg != 1 else W.make_workload(cfg)
        for r in range(len(wl.requests)):
            for l in (0, 1, wl.geom.n_layers - 1):
                kv.kvpool_validate_table(wl.layer_table(r, l), wl.nphys)
    kv.kvpool_validate_table(np.zeros(0, np.int32), 1)                       # K = 0 is valid
    kv.kvpool_validate_table(np.arange(64, dtype=np.int32)[::-1], 64)        # a full permutation
    for bad, nphys, word in (([0, 1, 64], 64, "outside"), ([0, -1], 64, "outside"), ([3, 5, 3], 64, "twice"), ([0, 1, 2], 2, "distinct")):
        with pytest.raises(kv.KvPoolError) as e:
            kv.kvpool_validate_table(np.array(bad, np.int32), nphys)
        assert e.value.code == kv.EINVAL and word in str(e.value)
    with pytest.raises(kv.KvPoolError) as e:
        kv.kvpool_validate_table(np.array([7, 9, 7], np.int32), 16)
    assert "entry 2" in str(e.value) and "block 7" in str(e.value)


def test_create_without_gpu_fails_loudly_with_ecuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(kv.KvPoolError) as e:
        kv.KvPool([1.0], [1 << 20], n_layers=1, n_kv_heads=1, head_dim=64)
    assert e.value.code == kv.ECUDA and "no CPU fallback" in str(e.value)


def test_create_argument_validation_precedes_cuda():
    for kwargs in (dict(n_layers=0, n_kv_heads=1, head_dim=64), dict(n_layers=1, n_kv_heads=1, head_dim=3, elem_bytes=1, block_tokens=1)):
        with pytest.raises(kv.KvPoolError) as e:
            kv.KvPool([1.0], [1 << 20], **kwargs)
        assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:
        kv.KvPool([1.0, -2.0], [1 << 20, 1 << 20], n_layers=1, n_kv_heads=1, head_dim=64)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:
        kv.KvPool([1.0], [0], n_layers=1, n_kv_heads=1, head_dim=64)
    assert e.value.code == kv.EINVAL
    for flags in (16, kv.DEV_HBM | kv.DEV_CUDA_HOSTALLOC, kv.DEV_HBM | kv.DEV_WRITE_COMBINED, kv.DEV_HBM | kv.DEV_NUMA_STRICT):      # unknown flag; HBM excludes host flags
        with pytest.raises(kv.KvPoolError) as e:
            kv.KvPool([1.0], [1 << 20], n_layers=1, n_kv_heads=1, head_dim=64, dev_flags=[flags])
        assert e.value.code == kv.EINVAL


def test_product_does_not_import_oracle_and_oracle_does_not_import_product():
    pkg = os.path.join(ROOT, "paper_2606_14779_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".hpp", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "kvpool_oracle" not in src and "liboracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_14779_b200" not in src.replace("paper_2606_14779_b200/", "") or f == "__init__.py"
            assert not re.search(r"^\s*(from|import)\s+paper_2606_14779_b200", src, re.M), f
            assert "kvpool.h" not in src, f


def test_plain_c_client_compiles_against_header_and_runs(tmp_path):
    """include/kvpool.h is valid C99 and the library is usable from C with nothing but pointers and sizes."""
    import subprocess
    exe = str(tmp_path / "c_abi_client")
    lib_dir = os.path.dirname(kv.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    os.path.join(ROOT, "tests", "c_abi_client.c"), "-o", exe, "-L", lib_dir, "-lkvpool", "-L", CUDA_LIB, "-lcudart", f"-Wl,-rpath,{lib_dir}"], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.splitlines()
    assert out[0] == "counts 2341 2341 1170 1170 585 585"
    od, _ = oracle.wrr(oracle.counts([4000, 4000, 2000, 2000, 1000, 1000], 64), 64)
    assert out[1] == "dev " + " ".join(str(int(d)) for d in od[:16])
    assert out[2].startswith('error "plan_weights') and out[3].startswith("kvpool")
    import ctypes                                              # the ctypes structs of the binding have the header's C layout
    assert out[4] == f"sizeof {ctypes.sizeof(kv.DeviceDesc)} {ctypes.sizeof(kv.Geometry)} {ctypes.sizeof(kv.Tuning)}"


def test_stripe_allocator_against_a_page_bitmap_model(tmp_path):
    """a4: the first-fit, coalescing allocator that hands placements their regions (csrc/placement.cpp, plain C++) against a
    bitmap model on random alloc/free sequences — aligned, disjoint, lowest fitting gap, exact accounting, full coalescing."""
    import subprocess
    exe = str(tmp_path / "stripe_alloc_check")
    subprocess.run(["g++", "-std=c++17", "-O1", "-Wall", "-Wextra", "-Werror", os.path.join(ROOT, "tests", "stripe_alloc_check.cpp"),
                    os.path.join(ROOT, "paper_2606_14779_b200", "csrc", "placement.cpp"), "-o", exe], check=True)
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.strip() == "stripe allocator ok", out.stdout


def test_plan_lba_range_matches_oracle_and_rejects_bad_arguments(golden_dir):
    """KV-passthrough's range length as the library computes it against the oracle's, on the hand-worked rows
    and on random sizes up to products beyond 2^64."""
    with open(os.path.join(golden_dir, "worked_lba_ranges.txt")) as f:
        rows = [[c.strip() for c in ln.split("|")] for ln in f if ln.strip() and not ln.startswith("#")]
    for n, kvs, sec, want, _ in rows:
        assert kv.kvpool_plan_lba_range(int(n), int(kvs), int(sec)) == int(want) == oracle.lba_range_len(int(n), int(kvs), int(sec))
    rng = np.random.default_rng(31)
    for _ in range(3000):
        n, kvs = int(rng.integers(0, 2 ** 33)), int(rng.integers(1, 2 ** 31))
        sec = int(rng.choice([512, 1024, 4096, 65536, 520, 1, 3]))
        assert kv.kvpool_plan_lba_range(n, kvs, sec) == oracle.lba_range_len(n, kvs, sec)
    assert kv.kvpool_plan_lba_range(2 ** 40, 2 ** 30, 4096) == 2 ** 58          # the product does not fit 64 bits, the result does
    with pytest.raises(kv.KvPoolError) as e:
        kv.kvpool_plan_lba_range(1, 1, 0)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                     # more than 2^64 sectors
        kv.kvpool_plan_lba_range(2 ** 63, 2 ** 63, 1)
    assert e.value.code == kv.EINVAL


@pytest.mark.parametrize("sector,kv_size,slots,lane_bytes", [(512, 1536, 333, 32 << 10), (4096, 1536, 333, 32 << 10), (512, 96, 777, 4096 + 2 * 512),
                                                            (4096, 65536, 21, 1 << 20), (4096, 5120, 57, 16 << 10)])
@pytest.mark.parametrize("engine", ["io_uring", "sync"])
def test_ssd_worker_stores_and_retrieves_lba_ranges_like_the_oracle(tmp_path, sector, kv_size, slots, lane_bytes, engine):
    """The host side of KV-passthrough (csrc/ssd_io.cpp: the device's worker thread, read-modify-write of edge sectors, zero
    padding, lane hand-over) without a GPU: tests/ssd_io_check.cpp plays the GPU's half of every command; the backing file
    must equal orc_ssd_direct_store's sector array — after the set has arrived in out-of-order instalments that start and
    end inside sectors — and the read-back must equal the set (orc_ssd_direct_retrieve of every KV cache)."""
    import subprocess
    exe = str(tmp_path / "ssd_io_check")
    csrc = os.path.join(ROOT, "paper_2606_14779_b200", "csrc")
    subprocess.run(["g++", "-std=c++17", "-O1", "-pthread", "-Wall", "-Wextra", "-Werror", os.path.join(ROOT, "tests", "ssd_io_check.cpp"),
                    os.path.join(csrc, "ssd_io.cpp"), "-o", exe], check=True)
    rng = np.random.default_rng(sector + kv_size)
    stripe = rng.integers(0, 256, size=slots * kv_size, dtype=np.uint8)
    first = 3
    n_sec = oracle.lba_range_len(slots, kv_size, sector)
    disk_path, fill = str(tmp_path / "disk.img"), 0xC3
    with open(disk_path, "wb") as f:
        f.write(bytes([fill]) * ((first + n_sec + 4) * sector))
    stripe.tofile(str(tmp_path / "stripe.bin"))
    cuts = sorted({0, slots, *[int(x) for x in rng.integers(1, slots, size=5)]})
    spans = [f"{a}:{b}" for a, b in zip(cuts, cuts[1:])]
    spans = [spans[i] for i in rng.permutation(len(spans))]                        # instalments arrive out of order
    out = subprocess.run([exe, disk_path, str(sector), str(kv_size), str(first), str(lane_bytes), "3", str(tmp_path / "stripe.bin"),
                          str(tmp_path / "out.bin")] + spans, capture_output=True, text=True, timeout=120,
                         env=dict(os.environ, KVPOOL_SSD_SYNC="1" if engine == "sync" else "0"))   # both engines of the worker
    assert out.returncode == 0 and out.stdout.startswith("ssd io ok"), out.stdout + out.stderr
    want = np.full((first + n_sec + 4) * sector, fill, dtype=np.uint8)
    assert oracle.ssd_direct_store(want, sector, first, stripe, kv_size) == n_sec
    assert np.array_equal(np.fromfile(disk_path, dtype=np.uint8), want)             # every sector, padding and neighbours included
    back = np.fromfile(str(tmp_path / "out.bin"), dtype=np.uint8)
    for s in [0, slots - 1] + [int(x) for x in rng.integers(0, slots, size=16)]:
        lba, off = oracle.ssd_location(first, s, kv_size, sector)
        assert np.array_equal(back[s * kv_size:(s + 1) * kv_size], oracle.ssd_direct_retrieve(want, sector, lba, off, kv_size))
    assert np.array_equal(back, stripe)
