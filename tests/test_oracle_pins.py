"""Pins for the CPU oracle (oracle/kvpool_oracle.c): it is checked against what the paper and the mathematics
fix, never against itself.  No GPU, no product code.  Each test says which plausible mistake it would catch.
"""
import itertools
import os
from decimal import Decimal, ROUND_HALF_UP
from fractions import Fraction
from math import floor

import numpy as np
import pytest

import oracle
from oracle import exact


def _golden_rows(golden_dir, name):
    with open(os.path.join(golden_dir, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                yield [c.strip() for c in line.split("|")]


# ------------------------------------------------------------------------------------------------
# geometry: values the paper prints
# ------------------------------------------------------------------------------------------------
def test_kv_bytes_matches_sizes_printed_in_paper(golden_dir):
    rows = list(_golden_rows(golden_dir, "paper_kv_sizes.txt"))
    assert len(rows) == 4
    for label, L, H, D, e, tokens, printed, decimals, _cite in rows:
        got = oracle.kv_bytes(int(L), int(H), int(D), int(e), int(tokens))
        gib = Decimal(got) / Decimal(2 ** 30)
        q = Decimal(1).scaleb(-int(decimals))
        assert gib.quantize(q, rounding=ROUND_HALF_UP) == Decimal(printed), label


def test_kv_bytes_matches_baseline_config_sizes():
    # BASELINE.json: 128 MiB @1K and 4 GiB @32K (LLaMA-8B), ~6 GiB (GPT-OSS-20B), ~12 GiB (Qwen3), bf16
    MiB, GiB = 2 ** 20, 2 ** 30
    assert oracle.kv_bytes(32, 8, 128, 2, 1024) == 128 * MiB
    assert oracle.kv_bytes(32, 8, 128, 2, 32768) == 4 * GiB
    assert oracle.kv_bytes(24, 8, 64, 2, 131072) == 6 * GiB
    assert oracle.kv_bytes(48, 4, 128, 2, 131072) == 12 * GiB
    assert sum(oracle.kv_bytes(32, 8, 128, 2, t) for t in (32768, 65536, 98304, 131072)) == 40 * GiB


# ------------------------------------------------------------------------------------------------
# weights: the single floating-point step
# ------------------------------------------------------------------------------------------------
def test_weights_are_bandwidth_in_integer_mb_per_s_round_half_up():
    b = [55.62, 57.26, 21.3, 63.0, 0.001, 2.0, 1.0, 12.3456]
    w = oracle.weights(b)
    for bi, wi in zip(b, w):
        # exact decimal value of the double, then round half up to an integer number of MB/s
        want = int((Decimal(bi) * 1000).quantize(Decimal(1), rounding=ROUND_HALF_UP))
        assert int(wi) == want
    with pytest.raises(ValueError):
        oracle.weights([1.0, 0.0])
    with pytest.raises(ValueError):
        oracle.weights([1.0, -3.0])
    with pytest.raises(ValueError):
        oracle.weights([0.0004])


# ------------------------------------------------------------------------------------------------
# counts: Eq. 1-2, Alg. 1 l.4-12
# ------------------------------------------------------------------------------------------------
def _random_cases(seed, n_cases, max_n=8, max_k=400, max_w=60000):
    rng = np.random.default_rng(seed)
    for _ in range(n_cases):
        n = int(rng.integers(1, max_n + 1))
        w = [int(x) for x in rng.integers(1, max_w + 1, size=n)]
        if rng.random() < 0.3:                       # force ties between weights
            w = [w[int(rng.integers(0, n))] if rng.random() < 0.5 else x for x in w]
        K = int(rng.integers(0, max_k + 1))
        yield w, K


def test_counts_invariants_exact_rational():
    """Catches: ceil/round instead of floor, remainder given to one device or to the wrong ones, float drift."""
    for w, K in _random_cases(1, 3000):
        c = [int(x) for x in oracle.counts(w, K)]
        W = sum(w)
        p = [Fraction(wi, W) for wi in w]
        assert sum(c) == K                                              # the constraint at PAPER.md:175
        fl = [floor(pi * K) for pi in p]
        assert all(ci in (f, f + 1) for ci, f in zip(c, fl))            # Eq. 2 with r_i in {0,1}
        assert all(abs(ci - pi * K) < 1 for ci, pi in zip(c, p))        # share within one block (north star)
        r = K - sum(fl)
        assert 0 <= r <= len(w) - 1 or (len(w) == 1 and r == 0)
        extras = {i for i in range(len(w)) if c[i] == fl[i] + 1}
        order = sorted(range(len(w)), key=lambda i: (-p[i], i))
        assert extras == set(order[:r])                                 # "devices with larger p_i"


def test_counts_unique_solution_by_brute_force():
    """Enumerate every vector with c_i in {floor, floor+1} and sum K whose +1 set is closed under 'larger p first';
    exactly one exists and the oracle returns it."""
    for w, K in _random_cases(2, 300, max_n=6, max_k=60, max_w=9):
        W = sum(w)
        fl = [(wi * K) // W for wi in w]
        # independent floor: compare against Fraction too
        assert fl == [floor(Fraction(wi, W) * K) for wi in w]
        sols = []
        for bits in itertools.product((0, 1), repeat=len(w)):
            if sum(fl) + sum(bits) != K:
                continue
            ok = True
            for i, j in itertools.permutations(range(len(w)), 2):
                # j got an extra but i did not although i has priority (larger p, or equal p and lower index)
                if bits[j] and not bits[i] and (w[i] > w[j] or (w[i] == w[j] and i < j)):
                    ok = False
            if ok:
                sols.append([f + b for f, b in zip(fl, bits)])
        assert len(sols) == 1
        assert [int(x) for x in oracle.counts(w, K)] == sols[0]


def test_counts_closed_forms():
    for n in (1, 2, 3, 4, 6, 8):
        for m in (0, 1, 5, 192, 1024):
            assert list(oracle.counts([7] * n, n * m)) == [m] * n           # equal weights, N | K
    assert list(oracle.counts([5], 12345)) == [12345]                       # one device takes everything
    # scaling all weights by a constant changes nothing (p_i is a ratio)
    for w, K in _random_cases(3, 200):
        assert list(oracle.counts(w, K)) == list(oracle.counts([3 * x for x in w], K))
    # huge weights and K: 128-bit product must not overflow (p*K computed exactly)
    w = [2 ** 40 + 1, 2 ** 40, 3]
    K = 2 ** 31 - 1
    c = [int(x) for x in oracle.counts(w, K)]
    assert sum(c) == K and all(abs(ci - Fraction(wi, sum(w)) * K) < 1 for ci, wi in zip(c, w))


def test_counts_and_wrr_hand_worked_examples(golden_dir):
    n_counts = n_wrr = 0
    for row in _golden_rows(golden_dir, "worked_placements.txt"):
        if row[0] == "counts":
            w = [int(x) for x in row[1].split(",")]
            want = [int(x) for x in row[3].split(",")]
            assert [int(x) for x in oracle.counts(w, int(row[2]))] == want, row
            n_counts += 1
        elif row[0] == "wrr":
            c = [int(x) for x in row[1].split(",")]
            dev, _ = oracle.wrr(c, sum(c))
            assert "".join(str(int(d)) for d in dev) == row[2], row
            n_wrr += 1
    assert n_counts >= 9 and n_wrr >= 6


# ------------------------------------------------------------------------------------------------
# weighted round-robin: Alg. 1 l.13-16
# ------------------------------------------------------------------------------------------------
def test_wrr_bijection_slot_order_and_prefix_fairness():
    """Catches: a block placed twice or never, slots not in enumeration order, bursty (first-fit) assignment."""
    for w, K in _random_cases(4, 1500):
        c = [int(x) for x in oracle.counts(w, K)]
        dev, slot = oracle.wrr(c, K)
        dev, slot = [int(x) for x in dev], [int(x) for x in slot]
        n = len(c)
        assert sorted(zip(dev, slot)) == [(i, s) for i in range(n) for s in range(c[i])]   # placed exactly once
        a = [0] * n
        for j in range(K):
            assert slot[j] == a[dev[j]]                                  # slots ascend with j within a device
            a[dev[j]] += 1
            for i in range(n):                                           # prefix fairness, both sides
                ideal = Fraction(c[i] * (j + 1), K)
                assert -1 < a[i] - ideal <= Fraction((n - 1) * c[i], K)


def test_wrr_equals_merge_of_sorted_ideal_times():
    """Independent algorithm: the k-th item of device i has ideal time k/c_i; a global sort of all
    (k/c_i, i) pairs (a library sort, no greedy loop) must give the same sequence."""
    for w, K in _random_cases(5, 600):
        c = [int(x) for x in oracle.counts(w, K)]
        dev, slot = oracle.wrr(c, K)
        keys = sorted((Fraction(k, c[i]), i, k - 1) for i in range(len(c)) for k in range(1, c[i] + 1))
        assert [int(d) for d in dev] == [i for _, i, _ in keys]
        assert [int(s) for s in slot] == [s for _, _, s in keys]


def test_wrr_closed_forms():
    for n in (1, 2, 4, 8):
        m = 24
        dev, slot = oracle.wrr([m] * n, n * m)
        assert list(dev) == [j % n for j in range(n * m)]                # equal counts: plain round-robin
        assert list(slot) == [j // n for j in range(n * m)]
    dev, _ = oracle.wrr([2 * 30, 30], 90)
    assert list(dev) == [0, 0, 1] * 30                                   # 2:1 with 3 | K
    dev, slot = oracle.wrr([17], 17)
    assert list(dev) == [0] * 17 and list(slot) == list(range(17))       # N = 1: identity
    dev, _ = oracle.wrr([0, 5, 0], 5)
    assert list(dev) == [1] * 5                                          # devices with c_i = 0 never chosen
    with pytest.raises(ValueError):
        oracle.wrr([2, 2], 5)                                            # counts must sum to K


def test_c_oracle_equals_exact_rational_statement():
    for w, K in _random_cases(6, 500, max_k=200):
        assert [int(x) for x in oracle.counts(w, K)] == exact.counts(w, K)
        c = exact.counts(w, K)
        d, s = oracle.wrr(c, K)
        d2, s2 = exact.wrr(c, K)
        assert [int(x) for x in d] == d2 and [int(x) for x in s] == s2


def test_place_applies_algorithm_per_layer():
    pls = oracle.place([2.0, 1.0], [64, 0, 8, 3])
    assert [list(p.counts) for p in pls] == [[43, 21], [0, 0], [6, 2], [2, 1]]   # 8*2/3 = 5.33 -> 5, 8/3 = 2.67 -> 2, 1 left -> dev 0
    assert [len(p.dev) for p in pls] == [64, 0, 8, 3]


# ------------------------------------------------------------------------------------------------
# gather / scatter: MEMSTORE and retrieval
# ------------------------------------------------------------------------------------------------
def _tiny_layer(rng, nphys, kvb):
    return rng.integers(0, 2 ** 16, size=(2, nphys, kvb // 2), dtype=np.uint16)


def test_offload_single_device_is_fancy_indexing():
    """N = 1: stripe == kv[:, table] with K and V interleaved per block (library routine)."""
    rng = np.random.default_rng(7)
    nphys, kvb, K = 37, 64, 23
    kv = _tiny_layer(rng, nphys, kvb)
    table = rng.permutation(nphys)[:K].astype(np.int32)
    pl = oracle.place([3.0], [K])[0]
    (stripe,) = oracle.offload_layer(kv, table, pl)
    want = np.stack([kv[0][table], kv[1][table]], axis=1)               # [K, 2, kvb/2]: K block then V block
    assert stripe.tobytes() == want.tobytes()
    # identity table over the whole pool: plain memcpy of K plane / V plane, interleaved per block
    table = np.arange(nphys, dtype=np.int32)
    pl = oracle.place([3.0], [nphys])[0]
    (stripe,) = oracle.offload_layer(kv, table, pl)
    assert stripe.tobytes() == np.stack([kv[0], kv[1]], axis=1).tobytes()


def test_retrieve_single_device_is_index_assignment():
    rng = np.random.default_rng(8)
    nphys, kvb, K = 29, 32, 11
    table = rng.permutation(nphys)[:K].astype(np.int32)
    pl = oracle.place([1.0], [K])[0]
    stripe = rng.integers(0, 256, size=K * 2 * kvb, dtype=np.uint8)
    out = np.full((2, nphys, kvb // 2), 0x7FC1, dtype=np.uint16)
    oracle.retrieve_layer(out, table, pl, [stripe])
    want = np.full((2, nphys, kvb // 2), 0x7FC1, dtype=np.uint16)
    pay = stripe.view(np.uint16).reshape(K, 2, kvb // 2)
    want[0][table] = pay[:, 0]
    want[1][table] = pay[:, 1]
    assert out.tobytes() == want.tobytes()


def test_offload_retrieve_match_brute_force_search():
    """Catches: K/V swapped, slot stride wrong, table applied on the wrong side, dev/slot transposed."""
    rng = np.random.default_rng(9)
    for _ in range(40):
        n = int(rng.integers(1, 6))
        bw = [float(x) for x in rng.integers(1, 9, size=n)]
        nphys = int(rng.integers(1, 40))
        K = int(rng.integers(0, nphys + 1))
        kvb = int(rng.choice([16, 48, 64]))
        kv = _tiny_layer(rng, nphys, kvb)
        table = rng.permutation(nphys)[:K].astype(np.int32)
        pl = oracle.place(bw, [K])[0]
        stripes = oracle.offload_layer(kv, table, pl)
        kb = [kv[0, p].tobytes() for p in range(nphys)]
        vb = [kv[1, p].tobytes() for p in range(nphys)]
        want = exact.offload_bruteforce(kb, vb, [int(t) for t in table], [int(d) for d in pl.dev],
                                        [int(s) for s in pl.slot], [int(c) for c in pl.counts])
        assert [s.tobytes() for s in stripes] == want
        # retrieve into poison, compare with the brute-force inverse
        out = np.full_like(kv, 0x7FC1)
        oracle.retrieve_layer(out, table, pl, stripes)
        kb2 = [np.full(kvb // 2, 0x7FC1, np.uint16).tobytes()] * nphys
        vb2 = list(kb2)
        kb2 = list(kb2)
        exact.retrieve_bruteforce(kb2, vb2, [int(t) for t in table], [int(d) for d in pl.dev],
                                  [int(s) for s in pl.slot], want, kvb)
        assert out[0].tobytes() == b"".join(kb2) and out[1].tobytes() == b"".join(vb2)


def test_round_trip_conservation_and_no_stray_writes():
    rng = np.random.default_rng(10)
    nphys, kvb, K = 96, 128, 64
    kv = _tiny_layer(rng, nphys, kvb)
    table = rng.permutation(nphys)[:K].astype(np.int32)
    pl = oracle.place([4, 4, 2, 2, 1, 1], [K])[0]
    stripes = oracle.offload_layer(kv, table, pl)
    # byte share per device within one block of its bandwidth share (north star invariant)
    P = 2 * kvb
    for s, wi in zip(stripes, [4, 4, 2, 2, 1, 1]):
        assert abs(Fraction(s.nbytes) - Fraction(wi, 14) * K * P) < P
    # conservation: multiset of payloads == multiset of the request's blocks
    pays = sorted(s[i * P:(i + 1) * P].tobytes() for s in stripes for i in range(s.nbytes // P))
    want = sorted(kv[0, t].tobytes() + kv[1, t].tobytes() for t in table)
    assert pays == want
    out = np.full_like(kv, 0x7FC1)
    oracle.retrieve_layer(out, table, pl, stripes)
    used = np.zeros(nphys, bool)
    used[table] = True
    assert np.array_equal(out[:, used], kv[:, used])                    # bit-for-bit round trip
    assert np.all(out[:, ~used] == 0x7FC1)                              # nothing else touched
    # worker-thread variant (Alg. 1 l.17) gives the same bytes
    stripes_mt = oracle.offload_layer(kv, table, pl, parallel=True)
    assert [a.tobytes() for a in stripes_mt] == [a.tobytes() for a in stripes]
    out_mt = np.full_like(kv, 0x7FC1)
    oracle.retrieve_layer(out_mt, table, pl, stripes, parallel=True)
    assert out_mt.tobytes() == out.tobytes()


def test_empty_layer_is_a_noop():
    kv = np.arange(2 * 4 * 8, dtype=np.uint16).reshape(2, 4, 8)
    pl = oracle.place([2.0, 1.0], [0])[0]
    stripes = oracle.offload_layer(kv, np.zeros(0, np.int32), pl)
    assert [s.nbytes for s in stripes] == [0, 0]
    out = kv.copy()
    oracle.retrieve_layer(out, np.zeros(0, np.int32), pl, stripes)
    assert np.array_equal(out, kv)


def test_retrieve_range_composes_and_touches_only_its_blocks():
    """Partial retrieval: (0, K) is the full retrieve; disjoint ranges compose to it; a range equals numpy index
    assignment of exactly its blocks; a prefix draws on every device within N-1 blocks of its share."""
    rng = np.random.default_rng(11)
    nphys, kvb, K = 120, 64, 90
    kv = _tiny_layer(rng, nphys, kvb)
    table = rng.permutation(nphys)[:K].astype(np.int32)
    w = [4, 4, 2, 2, 1, 1]
    pl = oracle.place(w, [K])[0]
    stripes = oracle.offload_layer(kv, table, pl)
    full = np.full_like(kv, 0x7FC1)
    oracle.retrieve_layer(full, table, pl, stripes)
    a = np.full_like(kv, 0x7FC1)
    oracle.retrieve_range(a, table, pl, stripes, 0, K)
    assert np.array_equal(a, full)
    b = np.full_like(kv, 0x7FC1)
    cuts = [0, 1, 17, 17, 50, 89, 90]
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        oracle.retrieve_range(b, table, pl, stripes, lo, hi - lo)
    assert np.array_equal(b, full)
    for first, n in ((0, 23), (23, 40), (89, 1), (40, 0)):
        c = np.full_like(kv, 0x7FC1)
        oracle.retrieve_range(c, table, pl, stripes, first, n)
        want = np.full_like(kv, 0x7FC1)
        want[:, table[first:first + n]] = kv[:, table[first:first + n]]      # library routine on exactly the range
        assert np.array_equal(c, want)
        for i, wi in enumerate(w):                                            # every device serves its share of the range
            took = int(np.sum(pl.dev[first:first + n] == i))
            assert abs(took - Fraction(int(pl.counts[i]) * n, K)) <= len(w) - 1 + 1


def test_offload_range_composes_and_writes_only_its_slots():
    """Partial offload (instalments of a request's blocks): (0, K) is the full offload; disjoint ranges
    compose to it in any order; a range equals numpy fancy indexing into exactly the slots Algorithm 1 gave its blocks
    (found here by an independent search over (dev, slot)); every other stripe byte keeps its fill."""
    rng = np.random.default_rng(13)
    nphys, kvb, K = 120, 64, 90
    kv = _tiny_layer(rng, nphys, kvb)
    table = rng.permutation(nphys)[:K].astype(np.int32)
    w = [4, 4, 2, 2, 1, 1]
    pl = oracle.place(w, [K])[0]
    full = oracle.offload_layer(kv, table, pl)
    P = 2 * kvb

    def filled():
        return [np.full(int(c) * P, 0xA5, dtype=np.uint8) for c in pl.counts]

    a = filled()
    oracle.offload_range(kv, table, pl, a, 0, K)
    assert all(np.array_equal(x, y) for x, y in zip(a, full))
    b = filled()
    cuts = [0, 1, 17, 17, 50, 89, 90]
    for lo, hi in reversed(list(zip(cuts[:-1], cuts[1:]))):               # instalments in reverse order
        oracle.offload_range(kv, table, pl, b, lo, hi - lo)
    assert all(np.array_equal(x, y) for x, y in zip(b, full))
    kv8 = kv.view(np.uint8).reshape(2, nphys, kvb)
    for first, n in ((0, 23), (23, 40), (89, 1), (40, 0)):
        c = filled()
        oracle.offload_range(kv, table, pl, c, first, n)
        want = filled()
        for i in range(len(w)):                                           # slot s of device i holds the unique j with (dev, slot) = (i, s)
            js = [j for j in range(first, first + n) if pl.dev[j] == i]
            for j in js:
                s_ = int(pl.slot[j])
                want[i][s_ * P:s_ * P + kvb] = kv8[0, table[j]]
                want[i][s_ * P + kvb:(s_ + 1) * P] = kv8[1, table[j]]
        assert all(np.array_equal(x, y) for x, y in zip(c, want)), (first, n)
    # what was offloaded in instalments comes back whole
    back = np.full_like(kv, 0x7FC1)
    oracle.retrieve_layer(back, table, pl, b)
    ref = np.full_like(kv, 0x7FC1)
    ref[:, table] = kv[:, table]
    assert np.array_equal(back, ref)


def test_checksum_closed_form_python_restatement_and_sensitivity():
    rng = np.random.default_rng(12)
    nphys, kvb, n = 19, 48, 11
    # constant words c: sum_idx c*(2*idx+1) = c * n_words^2
    c = 0x0123456789ABCDEF
    kv = np.full((2, nphys, kvb // 2), 0, dtype=np.uint16)
    kv.view(np.uint64)[...] = c
    table = rng.permutation(nphys)[:n].astype(np.int32)
    n_words = n * 2 * (kvb // 8)
    assert oracle.checksum(kv, table) == (c * n_words * n_words) % 2 ** 64
    # python big-int restatement on random data
    kv = _tiny_layer(rng, nphys, kvb)
    want, idx = 0, 0
    for j in range(n):
        for h in range(2):
            for w in kv[h, table[j]].view(np.uint64):
                want += int(w) * (2 * idx + 1)
                idx += 1
    assert oracle.checksum(kv, table) == want % 2 ** 64
    # swapping two table entries (two blocks trade places) or K with V changes it; an empty table sums to 0
    t2 = table.copy()
    t2[[0, 5]] = t2[[5, 0]]
    assert oracle.checksum(kv, t2) != oracle.checksum(kv, table)
    assert oracle.checksum(np.ascontiguousarray(kv[::-1]), table) != oracle.checksum(kv, table)
    assert oracle.checksum(kv, table[:0]) == 0


# ------------------------------------------------------------------------------------------------
# KV-passthrough: LBA range length, SSD_Direct_Store, GLT location, SSD_Direct_Retrieve
# ------------------------------------------------------------------------------------------------
def test_lba_range_length_hand_worked_values_and_the_definition_of_a_ceiling(golden_dir):
    rows = list(_golden_rows(golden_dir, "worked_lba_ranges.txt"))
    assert len(rows) == 10
    for n, kv, sec, want, _how in rows:
        assert oracle.lba_range_len(int(n), int(kv), int(sec)) == int(want), (n, kv, sec)
    # the defining property of ceil(x) for x = n*kv/sec, in exact rationals: len - 1 < x <= len
    # (a floor, a "+1 always" or a rounding to nearest each break one side of it)
    rng = np.random.default_rng(21)
    for _ in range(2000):
        n, kv = int(rng.integers(0, 5000)), int(rng.integers(1, 70000))
        sec = int(rng.choice([512, 520, 4096, 4160, 1, 7]))
        got, x = oracle.lba_range_len(n, kv, sec), Fraction(n * kv, sec)
        assert got - 1 < x <= got
    # no 64-bit overflow in set_size * kv_size (a 16 EiB product still divides exactly)
    assert oracle.lba_range_len(2 ** 40, 2 ** 30, 4096) == 2 ** 58


def test_ssd_direct_store_is_a_slice_assignment_of_the_sector_array_zero_padded():
    rng = np.random.default_rng(22)
    for kv, sec, n, first, sectors in [(96, 512, 17, 3, 16), (65536, 512, 5, 100, 800), (1536, 4096, 5, 1, 4), (48, 512, 1, 0, 1), (512, 512, 9, 7, 16)]:
        stripe = rng.integers(0, 256, size=n * kv, dtype=np.uint8)
        disk = np.full(sectors * sec, 0xA5, dtype=np.uint8)
        length = oracle.ssd_direct_store(disk, sec, first, stripe, kv)
        assert length == oracle.lba_range_len(n, kv, sec)
        rows = disk.reshape(sectors, sec)
        flat = rows[first:first + length].reshape(-1)
        assert np.array_equal(flat[:n * kv], stripe)                       # payloads back to back from the first sector on
        assert not flat[n * kv:].any()                                     # the rest of the last sector is zero
        assert (rows[:first] == 0xA5).all() and (rows[first + length:] == 0xA5).all()   # neighbours untouched
        if kv % sec == 0:                                                  # sector-multiple payloads: whole-sector copies, no padding
            assert length * sec == n * kv
    with pytest.raises(ValueError):                                        # a range that runs off the disk is refused, nothing written
        disk = np.full(4 * 512, 0xA5, dtype=np.uint8)
        oracle.ssd_direct_store(disk, 512, 3, np.zeros(2 * 512, dtype=np.uint8), 512)
    assert (disk == 0xA5).all()
    # the empty set writes nothing
    disk = np.full(4 * 512, 0xA5, dtype=np.uint8)
    assert oracle.ssd_direct_store(disk, 512, 2, np.zeros(0, dtype=np.uint8), 64) == 0 and (disk == 0xA5).all()


def test_ssd_location_and_direct_retrieve_find_every_kv_cache_by_its_byte_address():
    rng = np.random.default_rng(23)
    for kv, sec, n, first in [(96, 512, 40, 5), (65536, 4096, 6, 2), (1536, 4096, 9, 0), (512, 512, 12, 3), (700, 520, 11, 1)]:
        stripe = rng.integers(0, 256, size=n * kv, dtype=np.uint8)
        sectors = first + oracle.lba_range_len(n, kv, sec) + 2
        disk = np.full(sectors * sec, 0x5A, dtype=np.uint8)
        oracle.ssd_direct_store(disk, sec, first, stripe, kv)
        seen = set()
        for s in range(n):
            lba, off = oracle.ssd_location(first, s, kv, sec)
            # the location is the byte address of the payload, split into (sector, byte inside it): brute force over the
            # candidates instead of trusting the division
            want = [(a, b) for a in range(sectors) for b in range(sec) if a * sec + b == first * sec + s * kv]
            assert [(lba, off)] == want
            assert 0 <= off < sec and (off == 0 or kv % sec)
            seen.add((lba, off))
            assert np.array_equal(oracle.ssd_direct_retrieve(disk, sec, lba, off, kv), stripe[s * kv:(s + 1) * kv])
        assert len(seen) == n                                              # distinct KV caches, distinct locations
        if kv % sec == 0:                                                  # LBA advances by KV_size / sector_size per cache
            assert [oracle.ssd_location(first, s, kv, sec)[0] for s in range(n)] == [first + s * (kv // sec) for s in range(n)]


def test_ssd_store_then_retrieve_reproduces_an_offloaded_layer():
    # MEMSTORE's stripe order is what SSD_Direct_Store writes (Alg. 1 l.18 / l.21 differ only in the medium): store the
    # pinned orc_offload_layer's stripes on two "SSDs", read every KV cache back through its location, scatter it
    rng = np.random.default_rng(24)
    nphys, kvb, K, sec = 23, 96, 17, 512
    kv = _tiny_layer(rng, nphys, kvb)
    table = rng.permutation(nphys)[:K].astype(np.int32)
    pl = oracle.place([3.0, 1.0], [K])[0]
    stripes = oracle.offload_layer(kv, table, pl)
    disks, first = [], [4, 1]
    for i in range(2):
        d = np.full(64 * sec, 0xEE, dtype=np.uint8)
        assert oracle.ssd_direct_store(d, sec, first[i], stripes[i], 2 * kvb) == oracle.lba_range_len(int(pl.counts[i]), 2 * kvb, sec)
        disks.append(d)
    back = np.full_like(kv, 0x7FC1)
    for j in range(K):
        i, s = int(pl.dev[j]), int(pl.slot[j])
        payload = oracle.ssd_direct_retrieve(disks[i], sec, *oracle.ssd_location(first[i], s, 2 * kvb, sec), 2 * kvb).view(np.uint16)
        back[0, table[j]], back[1, table[j]] = payload[:kvb // 2], payload[kvb // 2:]
    ref = np.full_like(kv, 0x7FC1)
    ref[:, table] = kv[:, table]
    assert np.array_equal(back, ref)
