"""Exact-rational, pure-Python statement of the same method — TEST INFRASTRUCTURE, tiny inputs only.

A second, independent wording of what `kvpool_oracle.c` computes, in the paper's notation with
`fractions.Fraction` (no integer tricks, no cross-multiplication), plus an O(K^2) brute-force
gather/scatter.  tests/test_oracle_pins.py checks the C oracle against this and against the invariants
the paper states; nothing in the product imports it.
"""
from __future__ import annotations

from fractions import Fraction
from math import floor
from typing import List, Sequence, Tuple


def ratios(w: Sequence[int]) -> List[Fraction]:
    """Eq. 1: p_i = b_i / sum_j b_j."""
    total = sum(w)
    return [Fraction(wi, total) for wi in w]


def counts(w: Sequence[int], K: int) -> List[int]:
    """Eq. 2 and Alg. 1 l.4-12."""
    p = ratios(w)
    target = [floor(pi * K) for pi in p]
    remaining = K - sum(target)
    # "distributes the remainder to the devices with larger p_i": one each, largest p first, lower index on ties
    order = sorted(range(len(w)), key=lambda i: (-p[i], i))
    for i in order[:remaining]:
        target[i] += 1
    return target


def wrr(c: Sequence[int], K: int) -> Tuple[List[int], List[int]]:
    """Alg. 1 l.13-16 as smooth weighted round-robin (R3)."""
    a = [0] * len(c)
    dev, slot = [], []
    for _ in range(K):
        open_ = [i for i in range(len(c)) if a[i] < c[i]]
        i = min(open_, key=lambda i: (Fraction(a[i] + 1, c[i]), i))
        dev.append(i)
        slot.append(a[i])
        a[i] += 1
    return dev, slot


def offload_bruteforce(k_blocks: List[bytes], v_blocks: List[bytes], table: Sequence[int], dev: Sequence[int],
                       slot: Sequence[int], c: Sequence[int]) -> List[bytes]:
    """Stripe i, slot s holds K||V of the unique j with (dev[j], slot[j]) == (i, s) — found by search."""
    stripes = []
    for i in range(len(c)):
        parts = []
        for s in range(c[i]):
            js = [j for j in range(len(table)) if dev[j] == i and slot[j] == s]
            assert len(js) == 1, "every slot holds exactly one KV cache"
            parts.append(k_blocks[table[js[0]]] + v_blocks[table[js[0]]])
        stripes.append(b"".join(parts))
    return stripes


def retrieve_bruteforce(k_blocks: List[bytes], v_blocks: List[bytes], table: Sequence[int], dev: Sequence[int],
                        slot: Sequence[int], stripes: List[bytes], kvb: int) -> None:
    """Inverse: for every logical block j read its payload by (device, slot) and write physical block table[j]."""
    for j in range(len(table)):
        payload = stripes[dev[j]][slot[j] * 2 * kvb:(slot[j] + 1) * 2 * kvb]
        k_blocks[table[j]] = payload[:kvb]
        v_blocks[table[j]] = payload[kvb:]
