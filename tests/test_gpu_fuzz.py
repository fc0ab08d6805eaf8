"""Randomised choreography test: seeded random sequences of place / offload / re-offload / retrieve / range retrieve /
batched calls (half of the batched retrieves through kvpool_retrieve_layers_signal, with a consumer behind the per-layer
events) / release over ONE pool, several live placements each on its own stream, random pool flavours (host and
HBM-type devices), random paths and tuning (1-3 staging slots, small groups), no synchronisation between operations
except at checkpoints.  Everything the library overlaps — staging-slot recycling, per-device I/O streams, landed events,
region reuse after release — must still produce the oracle's bytes: every retrieve lands in a fresh poison-filled tensor
that is compared whole at the next checkpoint, and every live stripe is compared with the oracle's.  Between checkpoints
the host only enqueues (expected values are computed at the checkpoint), so the GPU works through a backlog of operations
that overlap as far as the library's events let them; dropping one of those waits makes this test fail."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import workloads as W

from parity_util import check_placement

pytestmark = pytest.mark.gpu

L, NPHYS, KMAX = 5, 1280, 1024
GEOM = dict(n_kv_heads=4, head_dim=128)         # kvb = 16 x 4 x 128 x 2 B = 16 KiB, P = 32 KiB: a 1024-block layer moves 32 MiB,
ELEMS = 16 * 4 * 128                            # 0.6 ms on the link, against ~50 us of host time per call: the GPU runs behind


@pytest.fixture(scope="module", autouse=True)
def _built():
    kvbuild.build()
    assert torch.cuda.is_available()
    kv.lib()


class Req:
    """One live placement: its stream, table, per-layer block counts and which source version each layer holds."""

    def __init__(self, rng, pool, bw, dev):
        self.stream = torch.cuda.Stream(device=dev)
        kinds = rng.integers(0, 4, size=L)
        self.bpl = [int((0, rng.integers(1, 9), rng.integers(300, KMAX + 1), rng.integers(KMAX // 2, KMAX + 1))[k]) for k in kinds]
        self.table_np = np.ascontiguousarray(rng.permutation(NPHYS)[:KMAX].astype(np.int32))
        with torch.cuda.stream(self.stream):
            self.table = torch.from_numpy(self.table_np).to(dev)
        self.stream.synchronize()
        self.pl = pool.place(self.bpl)
        self.opl = oracle.place(bw, self.bpl)
        check_placement(self.pl, self.opl)
        self.version = [None] * L                # source version in the pool, per layer
        self.stripes = {}                        # (layer, version) -> oracle stripes


@pytest.mark.timeout(600)
@pytest.mark.parametrize("seed,ssd", [(1, False), (2, False), (3, False), (4, False), (5, False), (6, False), (7, True), (8, True), (9, True)])
def test_random_sequences_match_the_oracle(seed, ssd, tmp_path):
    rng = np.random.default_rng(14779 + seed)
    dev = torch.device("cuda:0")
    n_dev = int(rng.integers(2, 6))
    bw = [float(rng.integers(1, 9)) for _ in range(n_dev)]
    flags = [kv.DEV_HBM if rng.random() < 0.3 else 0 for _ in range(n_dev)]
    flags[int(rng.integers(0, n_dev))] = 0                                     # at least one host device
    cap = 4 * L * KMAX * 2 * ELEMS * 2                                         # room for 4 placements on any one device
    # link groups (devices of one group share an I/O stream per direction) from a generator of their own, so that the
    # operation sequences of the seeds stay what they were before groups existed
    groups = [int(x) for x in np.random.default_rng(977 + seed).integers(0, 3, size=n_dev)]
    paths = [None] * n_dev
    if ssd:
        # one or two devices become SSD-type (files opened O_DIRECT; KV-passthrough): their shares travel
        # through bounce lanes handed between streams and a worker thread, with small commands so that lanes are recycled
        # while several requests on several streams are in flight
        pick = np.random.default_rng(555 + seed)
        for i in pick.permutation(n_dev)[:int(pick.integers(1, 3))]:
            flags[int(i)], paths[int(i)] = kv.DEV_SSD, str(tmp_path / f"ssd{int(i)}.img")
    pool = kv.KvPool(bw, [cap] * n_dev, n_layers=L, dev_flags=flags, link_groups=groups, paths=paths,
                     sector_bytes=[4096 if f == kv.DEV_SSD and seed % 2 else 0 if f != kv.DEV_SSD else 512 for f in flags], **GEOM)
    if ssd:
        pool.set_tuning(ssd_lanes=int(np.random.default_rng(seed).integers(1, 4)), ssd_chunk_bytes=int(np.random.default_rng(seed).choice([64 << 10, 1 << 20, 8 << 20])))
    src_np = [[rng.integers(0, 0x7F80, size=(2, NPHYS, ELEMS), dtype=np.uint16) for _ in range(L)] for _ in range(2)]
    src = [[torch.from_numpy(a.view(np.int16)).to(dev) for a in vs] for vs in src_np]
    torch.cuda.synchronize()
    kvb = ELEMS * 2
    pending = []                                                               # (dst tensor, expected numpy, description)
    reqs = []
    signal_rng = np.random.default_rng(4242 + seed)                            # (its own generator: the operation sequences of the seeds stay what they were)
    consumer = torch.cuda.Stream(device=dev)

    def stripes_of(r, l, v=None):
        v = r.version[l] if v is None else v
        if (l, v) not in r.stripes:
            r.stripes[(l, v)] = oracle.offload_layer(src_np[v][l], r.table_np[:r.bpl[l]], r.opl[l])
        return r.stripes[(l, v)]

    def expect(r, l, v, first=None, n=None):
        """The oracle's result of the retrieve just enqueued, computed later (at the checkpoint)."""
        def compute():
            want = W.poison_numpy((2, NPHYS, ELEMS))
            if first is None:
                oracle.retrieve_layer(want, r.table_np[:r.bpl[l]], r.opl[l], stripes_of(r, l, v))
            else:
                oracle.retrieve_range(want, r.table_np[:r.bpl[l]], r.opl[l], stripes_of(r, l, v), first, n)
            return want
        return compute

    def fresh_dst(r):
        with torch.cuda.stream(r.stream):
            return W.poison_torch((2, NPHYS, ELEMS), dev)

    def checkpoint():
        torch.cuda.synchronize()
        pool.synchronize()
        for dst, want, what in pending:
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), want()), what
        pending.clear()
        for r in reqs:
            for l in range(L):
                if r.version[l] is None or r.bpl[l] == 0:
                    continue
                want = stripes_of(r, l)
                for i in range(n_dev):
                    assert np.array_equal(r.pl.stripe(l, i), want[i]), ("stripe", seed, l, i)

    def random_setup():
        pool.set_path(int(rng.choice([kv.PATH_AUTO, kv.PATH_STAGED, kv.PATH_STAGED, kv.PATH_ZEROCOPY])))

    try:
        pool.set_tuning(stage_slots=int(rng.integers(1, 4)), group_bytes=int(rng.choice([1 << 20, 8 << 20, 64 << 20])),
                        auto_threshold_bytes=int(rng.choice([64 << 10, 1 << 20, 8 << 20])),
                        kernel=int(rng.integers(0, 2)), link_kernel=int(rng.integers(0, 2)),
                        stage_chunk_bytes=int(rng.choice([2 ** 64 - 1, 2 ** 64 - 1, 96 << 10, 1 << 20, 5 << 20])))   # off, or chunked staging
        pool.set_path(kv.PATH_STAGED)
        pool.reserve_staging(KMAX * 2 * kvb)                                   # zero-copy placements never shrink the ring
        for step in range(90):
            if len(reqs) < 3 and (not reqs or rng.random() < 0.25):
                reqs.append(Req(rng, pool, bw, dev))
                continue
            r = reqs[int(rng.integers(0, len(reqs)))]
            op = rng.random()
            random_setup()
            if op < 0.30:                                                      # offload / re-offload one layer
                l, v = int(rng.integers(0, L)), int(rng.integers(0, 2))
                pool.offload(r.pl, l, src[v][l][0], src[v][l][1], kvb, r.table, r.stream)
                r.version[l] = v
            elif op < 0.36:                                                    # re-offload of a range of a layer already in the pool
                l = int(rng.integers(0, L))
                if r.version[l] is None or r.bpl[l] < 2:
                    continue
                first = int(rng.integers(0, r.bpl[l])); n = int(rng.integers(1, r.bpl[l] - first + 1))
                v = int(rng.integers(0, 2))
                pool.offload_range(r.pl, l, first, n, src[v][l][0], src[v][l][1], kvb, r.table, r.stream)
                base = stripes_of(r, l)                                        # oracle: the range lands on top of what was there
                mixed = [x.copy() for x in base]
                oracle.offload_range(src_np[v][l], r.table_np[:r.bpl[l]], r.opl[l], mixed, first, n)
                r.version[l] = ("mix", step)
                r.stripes[(l, r.version[l])] = mixed
            elif op < 0.42:                                                    # batched offload of a run of layers
                a = int(rng.integers(0, L)); n = int(rng.integers(1, L - a + 1)); v = int(rng.integers(0, 2))
                pool.offload_layers(r.pl, a, [src[v][l][0] for l in range(a, a + n)], [src[v][l][1] for l in range(a, a + n)], kvb,
                                    [r.table] * n, r.stream)
                for l in range(a, a + n):
                    r.version[l] = v
            elif op < 0.62:                                                    # retrieve one layer
                l = int(rng.integers(0, L))
                if r.version[l] is None:
                    continue
                dst = fresh_dst(r)
                pool.retrieve(r.pl, l, dst[0], dst[1], kvb, r.table, r.stream)
                pending.append((dst, expect(r, l, r.version[l]), ("retrieve", seed, step, l)))
            elif op < 0.76:                                                    # partial retrieval
                l = int(rng.integers(0, L))
                if r.version[l] is None or r.bpl[l] == 0:
                    continue
                first = int(rng.integers(0, r.bpl[l])); n = int(rng.integers(0, r.bpl[l] - first + 1))
                dst = fresh_dst(r)
                pool.retrieve_range(r.pl, l, first, n, dst[0], dst[1], kvb, r.table, r.stream)
                pending.append((dst, expect(r, l, r.version[l], first, n), ("range", seed, step, l, first, n)))
            elif op < 0.88:                                                    # batched retrieve of a run of offloaded layers
                a = int(rng.integers(0, L)); n = 0
                while a + n < L and r.version[a + n] is not None:
                    n += 1
                if n == 0:
                    continue
                dsts = [fresh_dst(r) for _ in range(n)]
                if signal_rng.random() < 0.5:
                    # the same through kvpool_retrieve_layers_signal: a consumer stream that waits on NOTHING but the per-layer
                    # events snapshots each layer as soon as its event fires; the snapshots must hold the oracle's bytes (on the
                    # zero-copy path small requests move as one launch that raises a flag per layer, kernels.cuh)
                    ready = [torch.cuda.Event() for _ in range(n)]
                    pool.retrieve_layers_signal(r.pl, a, [d[0] for d in dsts], [d[1] for d in dsts], kvb, [r.table] * n, ready, r.stream)
                    for q, l in enumerate(range(a, a + n)):
                        consumer.wait_event(ready[q])
                        with torch.cuda.stream(consumer):
                            snap = dsts[q].clone()
                        pending.append((snap, expect(r, l, r.version[l]), ("retrieve_layers_signal snapshot", seed, step, l)))
                else:
                    pool.retrieve_layers(r.pl, a, [d[0] for d in dsts], [d[1] for d in dsts], kvb, [r.table] * n, r.stream)
                for q, l in enumerate(range(a, a + n)):
                    pending.append((dsts[q], expect(r, l, r.version[l]), ("retrieve_layers", seed, step, l)))
            elif op < 0.91:
                checkpoint()
            else:                                                              # release: the caller's stream work must be over
                r.stream.synchronize()
                checkpoint()
                r.pl.release()
                reqs.remove(r)
        checkpoint()
        for r in reqs:
            r.pl.release()
    finally:
        pool.destroy()
