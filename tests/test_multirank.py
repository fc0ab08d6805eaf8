"""World-size-2 gloo test (CPU) of the N>1 host logic: ranks shard heads / requests, place independently through the
C ABI's pure-host entry points, and agree without any data-path collective; timings reduce as max over ranks."""
import hashlib
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import sharding
from paper_2606_14779_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.make_workload(5)
        # tensor-parallel sharding: same blocks, fewer heads per rank -> identical maps, P shrinks by tp
        first, n_heads = sharding.shard_heads(wl.geom.n_kv_heads, world, rank)
        bw = [55.6, 55.1, 54.9, 55.3, 30.2, 30.1, 29.9, 30.0] if rank == 0 else [1.0] * 8
        bw = sharding.agree_on_bandwidth(bw)                      # a few bytes, once, off the data path
        w = kv.kvpool_plan_weights(bw)
        h = hashlib.sha256()
        for r in range(len(wl.requests)):
            for K in sorted(set(int(k) for k in wl.blocks_per_layer(r))):
                c, d, s = kv.kvpool_plan_layer(w, K)
                h.update(c.tobytes() + d.tobytes() + s.tobytes())
        digest = torch.from_numpy(np.frombuffer(h.digest(), dtype=np.uint8).copy())
        gathered = [torch.zeros_like(digest) for _ in range(world)]
        dist.all_gather(gathered, digest)
        same = all(torch.equal(g, gathered[0]) for g in gathered)
        # data-parallel sharding of the four requests + max-over-ranks timing
        mine = sharding.shard_requests(len(wl.requests), world, rank)
        t = sharding.max_over_ranks([10.0 + rank, 5.0 - rank])
        out_q.put((rank, same, first, n_heads, mine, t, [int(x) for x in w]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_place_identically_without_a_collective():
    kvbuild.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, same0, f0, n0, mine0, t0, w0), (r1, same1, f1, n1, mine1, t1, w1) = res
    assert same0 and same1                                   # both ranks derived bit-identical placement maps
    assert (f0, n0, f1, n1) == (0, 4, 4, 4)                  # 8 KV heads over tp=2
    assert mine0 == [0, 2] and mine1 == [1, 3]               # requests dealt round-robin, disjoint, complete
    assert t0 == t1 == [11.0, 5.0]                           # max over ranks
    assert w0 == w1 == [55600, 55100, 54900, 55300, 30200, 30100, 29900, 30000]


def test_sharding_helpers_reject_bad_arguments():
    with pytest.raises(ValueError):
        sharding.shard_heads(8, 3, 0)
    with pytest.raises(ValueError):
        sharding.shard_heads(8, 2, 2)
    assert sharding.shard_requests(5, 2, 1) == [1, 3]
    assert sharding.max_over_ranks([1.0, 2.0]) == [1.0, 2.0]  # no process group: identity
