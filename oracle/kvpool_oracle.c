/*
 * kvpool_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the unified-KV-pooling hot path computes,
 * written from the paper (/root/reference/PAPER.md, arxiv 2606.14779) and the readings of it listed
 * in DESIGN.md §4.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code, header, table or helper with paper_2606_14779_b200/csrc/ and
 * includes nothing from include/.
 *
 * Everything here is integer or byte work; there is no floating point beyond the one-time
 * quantisation of a measured bandwidth to an integer weight (reading R5), so parity with
 * the CUDA path is bit-exact.
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/):
 *   orc_kv_bytes            — the paper's own printed KV sizes
 *   orc_weights/orc_counts  — exact-rational invariants of Eq. 1-2 (Fractions), uniqueness by brute
 *                             force over all count vectors, closed forms, hand-worked examples
 *   orc_wrr                 — closed forms (equal weights, 2:1, N=1), bijection, prefix-fairness bound,
 *                             independent exact-rational restatement, hand-worked example
 *   orc_offload/orc_retrieve— N=1 reduces to numpy fancy indexing / index assignment, identity table
 *                             reduces to memcpy, O(K^2) brute-force search, round trip, conservation
 *   orc_retrieve_range      — (0, K) equals orc_retrieve_layer; disjoint ranges compose to the full retrieve; numpy
 *                             index assignment on the range; nothing outside the range's physical blocks is written
 *   orc_offload_range       — (0, K) equals orc_offload_layer; disjoint ranges compose to the full offload; numpy fancy
 *                             indexing into the range's slots; stripe bytes outside the range's slots keep their fill
 *   orc_checksum            — closed form n_words^2 * c for constant words, python big-int restatement, sensitivity
 *                             to swapping two blocks
 *   orc_lba_range_len       — the paper's own formula against hand-worked values (tests/golden/
 *                             worked_lba_ranges.txt), the defining inequality of a ceiling, exact rationals
 *   orc_ssd_direct_store / orc_ssd_direct_retrieve / orc_ssd_location
 *                           — numpy slicing of the sector array, sector-multiple KV sizes reduce to whole-sector
 *                             copies, zero padding and untouched neighbours, brute-force byte addresses, round trip
 *   stripe offsets inside a pool buffer and the FIRST LBA of a range: PARITY UNPINNED (allocator detail; not produced here).
 *
 * Build: gcc -O2 -shared -fPIC -pthread -o liboracle.so kvpool_oracle.c   (oracle/__init__.py does it)
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>
#include <pthread.h>

#define ORC_MAX_DEV 64

/* ---- geometry --------------------------------------------------------------------------------
 * KV bytes of a model at a context length: one K and one V vector of H_kv*D elements per layer per
 * token.  PAPER.md:28 (LLaMA-3.1-405B FP32: 0.98 GB @1K, 123.05 GB @128K) and PAPER.md:321
 * (ref. [13], LLaMA-3.1-70B FP16: 0.313 GB @1K, 39.06 GB @128K) print values of this formula. */
uint64_t orc_kv_bytes(uint64_t n_layers, uint64_t n_kv_heads, uint64_t head_dim, uint64_t elem_bytes,
                      uint64_t tokens) {
    return 2u * n_layers * n_kv_heads * head_dim * elem_bytes * tokens;
}

/* ---- Eq. 1: placement ratios -----------------------------------------------------------------
 * p_i = b_i / sum_j b_j.  Kept exact: b_i is quantised ONCE to an integer weight
 * w_i = floor(b_i*1000 + 0.5) (bandwidth in MB/s, R5) and p_i is the rational w_i / W.
 * Returns 0, or -1 if some weight would be < 1 (bandwidth must be positive). */
int orc_weights(const double *bandwidth_gbps, uint32_t n, uint64_t *w) {
    for (uint32_t i = 0; i < n; ++i) {
        double x = bandwidth_gbps[i] * 1000.0 + 0.5;
        if (!(x >= 1.0) || x > 1.0e15) return -1;
        w[i] = (uint64_t)x;              /* truncation of a positive value = floor */
    }
    return 0;
}

/* ---- Eq. 2 / Algorithm 1 lines 4-12: target counts -------------------------------------------
 * target_i = floor(p_i * K)                                   (Alg. 1 l.5,  PAPER.md:198)
 * remaining = K - sum_i target_i                              (Alg. 1 l.8,  PAPER.md:202)
 * the remaining ones go, one each, to the devices with the larger p_i      (
 * DESIGN.md R2: ties broken by lower device index). */
int orc_counts(const uint64_t *w, uint32_t n, uint64_t K, uint32_t *count) {
    if (n == 0 || n > ORC_MAX_DEV) return -1;
    unsigned __int128 W = 0;
    for (uint32_t i = 0; i < n; ++i) { if (w[i] == 0) return -1; W += w[i]; }
    uint64_t assigned = 0;
    for (uint32_t i = 0; i < n; ++i) {
        unsigned __int128 prod = (unsigned __int128)w[i] * K;
        count[i] = (uint32_t)(prod / W);
        assigned += count[i];
    }
    uint64_t remaining = K - assigned;
    /* order devices by (p_i descending, index ascending): plain selection, N is tiny */
    uint8_t taken[ORC_MAX_DEV] = {0};
    for (uint64_t r = 0; r < remaining; ++r) {
        int best = -1;
        for (uint32_t i = 0; i < n; ++i) {
            if (taken[i]) continue;
            if (best < 0 || w[i] > w[best]) best = (int)i;
        }
        if (best < 0) return -1;         /* cannot happen: remaining <= n-1 */
        taken[best] = 1;
        count[best] += 1;
    }
    return 0;
}

/* ---- Algorithm 1 lines 13-16: partition in enumeration order ---------------------------------
 * "for all kv in K: select u_i such that |offload_set_i| < target_i", made
 * deterministic as a smooth weighted round-robin (R3): the next KV cache goes to the
 * device whose set would be least full relative to its target after receiving it, i.e. the i that
 * minimises (a_i + 1) / c_i among devices with a_i < c_i; ties to the lowest index.  Fractions are
 * compared exactly by cross-multiplication.  dev[j] = chosen device, slot[j] = its position in
 * that device's offload set (the order MEMSTORE lays the set out in, Alg. 1 l.18). */
int orc_wrr(const uint32_t *count, uint32_t n, uint64_t K, uint32_t *dev, uint32_t *slot) {
    uint64_t a[ORC_MAX_DEV];
    if (n == 0 || n > ORC_MAX_DEV) return -1;
    for (uint32_t i = 0; i < n; ++i) a[i] = 0;
    for (uint64_t j = 0; j < K; ++j) {
        int best = -1;
        for (uint32_t i = 0; i < n; ++i) {
            if (a[i] >= count[i]) continue;
            if (best < 0) { best = (int)i; continue; }
            /* (a_i+1)/c_i < (a_best+1)/c_best  <=>  (a_i+1)*c_best < (a_best+1)*c_i */
            unsigned __int128 lhs = (unsigned __int128)(a[i] + 1) * count[best];
            unsigned __int128 rhs = (unsigned __int128)(a[best] + 1) * count[i];
            if (lhs < rhs) best = (int)i;
        }
        if (best < 0) return -1;         /* counts do not sum to K */
        dev[j] = (uint32_t)best;
        slot[j] = (uint32_t)a[best];
        a[best] += 1;
    }
    return 0;
}

/* ---- Algorithm 1 lines 17-19, MEM branch: MEMSTORE --------------------------------------------
 * Offload one layer: KV cache j (logical block j of the request) lives in the paged layout at
 * physical block table[j]: K block = kvb bytes at k_plane + table[j]*stride, V block likewise in
 * v_plane.  Its pool payload is K block then V block (P = 2*kvb bytes, R6/R7), stored at
 * slot[j] of device dev[j]'s stripe for this layer.  stripes[i] points at c_i*P bytes. */
void orc_offload_layer(const uint8_t *k_plane, const uint8_t *v_plane, uint64_t stride, uint64_t kvb,
                       const int32_t *table, uint64_t K, const uint32_t *dev, const uint32_t *slot,
                       uint8_t *const *stripes) {
    for (uint64_t j = 0; j < K; ++j) {
        uint8_t *dst = stripes[dev[j]] + (uint64_t)slot[j] * 2u * kvb;
        memcpy(dst, k_plane + (uint64_t)table[j] * stride, kvb);
        memcpy(dst + kvb, v_plane + (uint64_t)table[j] * stride, kvb);
    }
}

/* ---- KV retrieval: the inverse ---------------------------------------------
 * Look up each KV cache's (device, location), read it by pointer, write it back to the paged layout
 * at physical block table[j].  Nothing else in the destination is touched. */
void orc_retrieve_layer(uint8_t *k_plane, uint8_t *v_plane, uint64_t stride, uint64_t kvb,
                        const int32_t *table, uint64_t K, const uint32_t *dev, const uint32_t *slot,
                        const uint8_t *const *stripes) {
    for (uint64_t j = 0; j < K; ++j) {
        const uint8_t *src = stripes[dev[j]] + (uint64_t)slot[j] * 2u * kvb;
        memcpy(k_plane + (uint64_t)table[j] * stride, src, kvb);
        memcpy(v_plane + (uint64_t)table[j] * stride, src + kvb, kvb);
    }
}

/* ---- partial retrieval -------------------------------------------------------------------------
 * "When a decoding step requests offloaded KV caches, the allocator first looks up their GLT entries"
 * (PAPER.md:241): the request may name any subset; here a contiguous range [first, first+n) of the
 * layer's logical blocks.  Same per-block procedure as orc_retrieve_layer, restricted to the range. */
void orc_retrieve_range(uint8_t *k_plane, uint8_t *v_plane, uint64_t stride, uint64_t kvb, const int32_t *table,
                        uint64_t first, uint64_t n, const uint32_t *dev, const uint32_t *slot,
                        const uint8_t *const *stripes) {
    for (uint64_t j = first; j < first + n; ++j) {
        const uint8_t *src = stripes[dev[j]] + (uint64_t)slot[j] * 2u * kvb;
        memcpy(k_plane + (uint64_t)table[j] * stride, src, kvb);
        memcpy(v_plane + (uint64_t)table[j] * stride, src + kvb, kvb);
    }
}

/* ---- partial offload ----------------------------------------------------------------------------
 * "At decoding step t, let K(t) denote the set of KV caches that must be offloaded": a
 * request's blocks reach the pool in instalments.  Here an instalment is a contiguous range
 * [first, first+n) of the layer's logical blocks, stored at the places Algorithm 1 gave them when the
 * layer was placed; same per-block MEMSTORE as orc_offload_layer, nothing outside the range's slots is
 * written. */
void orc_offload_range(const uint8_t *k_plane, const uint8_t *v_plane, uint64_t stride, uint64_t kvb, const int32_t *table,
                       uint64_t first, uint64_t n, const uint32_t *dev, const uint32_t *slot, uint8_t *const *stripes) {
    for (uint64_t j = first; j < first + n; ++j) {
        uint8_t *dst = stripes[dev[j]] + (uint64_t)slot[j] * 2u * kvb;
        memcpy(dst, k_plane + (uint64_t)table[j] * stride, kvb);
        memcpy(dst + kvb, v_plane + (uint64_t)table[j] * stride, kvb);
    }
}

/* ---- consumer stand-in checksum (not in the paper; defined in include-free words here) ---------------
 * sum over logical blocks j < n, halves h (0 = K block, 1 = V block), 64-bit little-endian words i of
 *     word(j,h,i) * (2*idx + 1)  mod 2^64,   idx = (j*2 + h)*(kvb/8) + i
 * where the blocks are read through the table: physical block table[j].  Order-independent (a sum),
 * position-sensitive (odd multipliers), so any misplaced, swapped or stale block changes it. */
uint64_t orc_checksum(const uint8_t *k_plane, const uint8_t *v_plane, uint64_t stride, uint64_t kvb,
                      const int32_t *table, uint64_t n) {
    uint64_t sum = 0, words = kvb / 8;
    for (uint64_t j = 0; j < n; ++j)
        for (uint64_t h = 0; h < 2; ++h) {
            const uint8_t *blk = (h ? v_plane : k_plane) + (uint64_t)table[j] * stride;
            for (uint64_t i = 0; i < words; ++i) {
                uint64_t w;
                memcpy(&w, blk + 8 * i, 8);
                sum += w * (2 * ((j * 2 + h) * words + i) + 1);
            }
        }
    return sum;
}

/* ---- "for all u_i in U in parallel" (Alg. 1 l.17; "each pool device has its own worker thread",
 * PAPER.md:177): the same two procedures with one worker thread per pool device, each handling the
 * KV caches assigned to its device.  Used only as the timed CPU baseline. */
typedef struct {
    int retrieve;
    uint32_t me;
    uint8_t *k_plane, *v_plane;
    uint64_t stride, kvb, K;
    const int32_t *table;
    const uint32_t *dev, *slot;
    uint8_t *const *stripes;
} orc_job;

static void *orc_worker(void *arg) {
    orc_job *jb = (orc_job *)arg;
    for (uint64_t j = 0; j < jb->K; ++j) {
        if (jb->dev[j] != jb->me) continue;
        uint8_t *s = jb->stripes[jb->me] + (uint64_t)jb->slot[j] * 2u * jb->kvb;
        uint8_t *k = jb->k_plane + (uint64_t)jb->table[j] * jb->stride;
        uint8_t *v = jb->v_plane + (uint64_t)jb->table[j] * jb->stride;
        if (jb->retrieve) { memcpy(k, s, jb->kvb); memcpy(v, s + jb->kvb, jb->kvb); }
        else              { memcpy(s, k, jb->kvb); memcpy(s + jb->kvb, v, jb->kvb); }
    }
    return NULL;
}

int orc_layer_parallel(int retrieve, uint8_t *k_plane, uint8_t *v_plane, uint64_t stride, uint64_t kvb,
                       const int32_t *table, uint64_t K, const uint32_t *dev, const uint32_t *slot,
                       uint8_t *const *stripes, uint32_t n) {
    pthread_t th[ORC_MAX_DEV];
    orc_job jb[ORC_MAX_DEV];
    if (n == 0 || n > ORC_MAX_DEV) return -1;
    for (uint32_t i = 0; i < n; ++i) {
        orc_job t = {retrieve, i, k_plane, v_plane, stride, kvb, K, table, dev, slot, stripes};
        jb[i] = t;
        if (pthread_create(&th[i], NULL, orc_worker, &jb[i]) != 0) return -1;
    }
    for (uint32_t i = 0; i < n; ++i) pthread_join(th[i], NULL);
    return 0;
}

/* ---- KV-passthrough, SSD branch of Algorithm 1 (l.20-21) and of the retrieval -----------
 * The SSD is an array of sectors addressed by logical block address (LBA): `disk` holds disk_sectors * sector_size
 * bytes, sector x at disk + x*sector_size.
 *
 * SSD_Direct_Store: "allocates a contiguous LBA range on the target device and writes the KV caches to that range ...
 * The LBA range length is ceil(|offload_set_i| * KV_size / sector_size) blocks". */
uint64_t orc_lba_range_len(uint64_t set_size, uint64_t kv_size, uint64_t sector_size) {
    unsigned __int128 bytes = (unsigned __int128)set_size * kv_size;
    uint64_t len = (uint64_t)(bytes / sector_size);
    if (bytes % sector_size) len += 1;          /* ceiling */
    return len;
}

/* The offload set (already in the order MEMSTORE would lay it out: slot 0, 1, ... — `set` holds set_size payloads of
 * kv_size bytes) is written to the range starting at first_lba, payloads back to back; what is left of the last sector
 * is zero (the paper does not say what fills it: DESIGN.md R18).  Sectors outside the range are not touched.  Returns
 * the range length in sectors, or UINT64_MAX if the range does not fit the disk. */
uint64_t orc_ssd_direct_store(uint8_t *disk, uint64_t disk_sectors, uint64_t sector_size, uint64_t first_lba,
                              const uint8_t *set, uint64_t set_size, uint64_t kv_size) {
    uint64_t len = orc_lba_range_len(set_size, kv_size, sector_size);
    if (first_lba > disk_sectors || len > disk_sectors - first_lba) return UINT64_MAX;
    uint8_t *at = disk + first_lba * sector_size;
    uint64_t bytes = set_size * kv_size;
    for (uint64_t s = 0; s < set_size; ++s) memcpy(at + s * kv_size, set + s * kv_size, kv_size);
    memset(at + bytes, 0, len * sector_size - bytes);
    return len;
}

/* "The resulting LBA information is returned to the bandwidth-aware KV allocator and stored in the GLT";
 * Table I: location = LBA for type SSD.  KV cache number `slot` of a set stored at first_lba starts in sector
 * first_lba + floor(slot*KV_size / sector_size), at byte (slot*KV_size) mod sector_size of that sector (0 whenever
 * KV_size is a multiple of the sector size, as for every model shape of the paper; R18). */
void orc_ssd_location(uint64_t first_lba, uint64_t slot, uint64_t kv_size, uint64_t sector_size, uint64_t *lba,
                      uint64_t *byte_in_sector) {
    unsigned __int128 off = (unsigned __int128)slot * kv_size;
    *lba = first_lba + (uint64_t)(off / sector_size);
    *byte_in_sector = (uint64_t)(off % sector_size);
}

/* SSD_Direct_Retrieve: "reads back a KV cache from SSD using the device_idx and location fields stored in the GLT"
 * (PAPER.md:185): kv_size bytes starting at (lba, byte_in_sector). */
void orc_ssd_direct_retrieve(const uint8_t *disk, uint64_t sector_size, uint64_t lba, uint64_t byte_in_sector,
                             uint8_t *payload_out, uint64_t kv_size) {
    memcpy(payload_out, disk + lba * sector_size + byte_in_sector, kv_size);
}
