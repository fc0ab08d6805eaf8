"""kvpool_pack_static — the pack for callers that cannot allocate GPU memory (code inside a serving engine that has given
HBM to its own KV allocator and must not stall on cudaMalloc): its maps sit in a fixed array inside the library instead
of in memory kvpool_place allocates.  Checked here against the pooled path it stands in for (kvpool_place + kvpool_pack)
and against the oracle, byte for byte (the tolerance of every test in this suite: none — byte moves only), on calls
that follow each other on one stream and therefore reuse the array while it still holds the previous call's maps.

The file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call then does the per-GPU look-up of the array) and after the other
tests (the library is loaded already, the array may hold anything)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import workloads as W

from parity_util import make_pool

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    kvbuild.build()
    assert torch.cuda.is_available()
    kv.lib()                                    # raises if libkvpool.so is missing: no fallback


@pytest.mark.parametrize("config,scale,n_layers", [(4, 1 / 16, 2), (3, 1 / 16, 4), (1, 1, 2)])
def test_pack_static_equals_pooled_pack_on_calls_in_a_row(config, scale, n_layers):
    """Every layer is packed twice: by kvpool_pack through a placement, and by kvpool_pack_static — the static calls
    issued back to back on one stream, nothing but stream order between them.  Config 3 alternates layers of 8 and 512
    blocks over four equal devices, so a call finds the longer maps of the call before it in the array; config 4 has the
    heterogeneous weights 4:4:2:2:1:1; config 1 two devices 2:1."""
    wl = W.make_workload(config, scale=scale, n_layers=n_layers)
    g = wl.geom
    bw = list(wl.default_weights())
    w = kv.kvpool_plan_weights(bw)
    bpl = wl.blocks_per_layer(0)
    opl = oracle.place(bw, bpl)
    stream = torch.cuda.Stream()
    pool = make_pool(wl)
    try:
        pl = pool.place(bpl)
        assert np.array_equal(pool.weights(), w)
        tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).cuda() for l in range(g.n_layers)]
        srcs = [W.kv_layer_torch(wl, l, "cuda:0") for l in range(g.n_layers)]
        pooled = [torch.zeros(int(bpl[l]) * g.payload, dtype=torch.uint8, device="cuda:0") for l in range(g.n_layers)]
        static = [torch.full((int(bpl[l]) * g.payload,), 0xA5, dtype=torch.uint8, device="cuda:0") for l in range(g.n_layers)]
        torch.cuda.synchronize()
        for rounds in range(2):                 # the second round starts from the array as the first left it
            for l in range(g.n_layers):
                kv.kvpool_pack_static(w, int(bpl[l]), srcs[l][0], srcs[l][1], g.kvb, tables[l], static[l], n_kv_heads=g.n_kv_heads,
                                      head_dim=g.head_dim, block_tokens=g.block_tokens, elem_bytes=g.elem_bytes, stream=stream)
        for l in range(g.n_layers):
            pool.pack(pl, l, srcs[l][0], srcs[l][1], g.kvb, tables[l], pooled[l])
        torch.cuda.synchronize()
        for l in range(g.n_layers):
            assert torch.equal(static[l], pooled[l]), f"layer {l}: static pack differs from the pooled pack"
            want = np.concatenate(oracle.offload_layer(W.kv_layer_numpy(wl, l), wl.layer_table(0, l), opl[l]))
            assert np.array_equal(static[l].cpu().numpy(), want), f"layer {l}: static pack differs from the oracle"
        pl.release()
    finally:
        pool.destroy()


def test_pack_static_at_its_largest_layer_and_refusal_beyond_it():
    """K = KVPOOL_STATIC_MAX_BLOCKS fills the array to its last entry (2 KiB K blocks: 128 MiB packed) and still equals the
    pooled pack; one block more is refused with EINVAL and a message that names the limit, and nothing is written."""
    K = kv.STATIC_MAX_BLOCKS
    heads, dim = 1, 64
    kvb = 16 * heads * dim * 2
    bw = [5.0, 3.0, 1.0]
    w = kv.kvpool_plan_weights(bw)
    gen = torch.Generator(device="cuda:0").manual_seed(7)
    src = torch.randint(0, 256, (2, K + 1, kvb), dtype=torch.uint8, device="cuda:0", generator=gen)
    table = torch.randperm(K + 1, device="cuda:0", generator=gen).to(torch.int32)
    static = torch.zeros(K * 2 * kvb, dtype=torch.uint8, device="cuda:0")
    pooled = torch.zeros_like(static)
    pool = kv.KvPool(bw, [K * 2 * kvb] * 3, n_layers=1, n_kv_heads=heads, head_dim=dim)
    try:
        pl = pool.place([K])
        for _ in range(2):
            kv.kvpool_pack_static(w, K, src[0], src[1], kvb, table, static, n_kv_heads=heads, head_dim=dim)
        pool.pack(pl, 0, src[0], src[1], kvb, table, pooled)
        torch.cuda.synchronize()
        assert torch.equal(static, pooled)
        counts, dev, slot = kv.kvpool_plan_layer(w, K)
        start = np.concatenate(([0], np.cumsum(counts)[:-1]))
        unit = (start[dev] + slot).astype(np.int64)          # where logical block j lands in the packed buffer
        got = static.view(K, 2, kvb).cpu().numpy()
        tab = table.cpu().numpy()
        srcn = src.cpu().numpy()
        for j in (0, 1, K // 2, K - 1):
            assert np.array_equal(got[unit[j], 0], srcn[0, tab[j]]) and np.array_equal(got[unit[j], 1], srcn[1, tab[j]])
        pl.release()
    finally:
        pool.destroy()
    before = static.clone()
    with pytest.raises(kv.KvPoolError) as err:
        kv.kvpool_pack_static(w, K + 1, src[0], src[1], kvb, table, static, n_kv_heads=heads, head_dim=dim)
    assert err.value.code == kv.EINVAL and "KVPOOL_STATIC_MAX_BLOCKS" in str(err.value)
    torch.cuda.synchronize()
    assert torch.equal(static, before)
    kv.kvpool_pack_static(w, 0, None, None, kvb, None, None, n_kv_heads=heads, head_dim=dim)   # an empty layer is a no-op
