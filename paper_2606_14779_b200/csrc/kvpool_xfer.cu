// libkvpool.so, part 2 of 3: the hot path (a5-a9) — per-layer, block-range and batched offload / retrieve over CUDA streams and
// events: the staged path (staging ring, copy engines, device-major chunks), the zero-copy and hybrid paths, kvpool_set_tables,
// and the in-device halves kvpool_pack / kvpool_unpack.
#include "kvpool_internal.hpp"

using namespace kvp;

extern "C" {


// Which blocks of a layer are in the pool (kvpool_offload_range fills a layer in instalments).
static void mark_offloaded(LayerState& L, uint32_t first, uint32_t n) {
  const uint64_t K = L.map->K;
  if (L.offloaded) return;
  if (n == K) { L.offloaded = true; L.have.clear(); return; }
  if (L.have.empty()) L.have.assign((K + 63) / 64, 0);
  for (uint32_t j = first; j < first + n; ++j) L.have[j >> 6] |= 1ull << (j & 63);
  uint64_t total = 0;
  for (uint64_t w : L.have) total += static_cast<uint64_t>(__builtin_popcountll(w));
  if (total == K) { L.offloaded = true; L.have.clear(); }
}
static bool is_offloaded(const LayerState& L, uint32_t first, uint32_t n) {
  if (L.offloaded) return true;
  if (L.have.empty()) return false;
  for (uint32_t j = first; j < first + n; ++j)
    if (!(L.have[j >> 6] >> (j & 63) & 1ull)) return false;
  return true;
}

// Slots of device i that hold logical blocks [first, first+n): a contiguous range because slots ascend with j.
static void slot_range(const LayerMap& m, uint32_t i, uint32_t first, uint32_t n, uint32_t* lo, uint32_t* hi) {
  if (first == 0 && n == m.K) { *lo = 0; *hi = m.counts[i]; return; }
  const auto b = m.order.begin() + m.start[i], e = b + m.counts[i];
  *lo = static_cast<uint32_t>(std::lower_bound(b, e, first) - b);
  *hi = static_cast<uint32_t>(std::lower_bound(b, e, first + n) - b);
}

// Blocks one staging slot can take: the slot's size, capped by tune.stage_chunk_bytes (layers larger than that travel
// in chunks of consecutive logical blocks, so the staging ring does not grow with the context length).
static uint64_t blocks_per_slot(const kvpool* p) {
  const uint64_t cap = p->tune.stage_chunk_bytes ? std::max<uint64_t>(p->tune.stage_chunk_bytes, p->payload) : ~0ull;
  return std::min(p->slot_bytes, cap) / p->payload;
}

// One chunk [first, first+n) of a layer through a staging slot.  The slot is compact: device 0's share of the chunk,
// then device 1's, ...; pool_base[i] is displaced so that slot index s of device i lands on its place in that share.
struct ChunkPlan {
  uint32_t lo[KVPOOL_MAX_DEVICES], hi[KVPOOL_MAX_DEVICES];
  uint64_t off[KVPOOL_MAX_DEVICES];  // byte offset of device i's share inside the slot
  uint64_t host_bytes = 0;           // what the chunk moves to / from host-memory devices
  bool host_blocks = false, hbm_blocks = false, ssd_blocks = false;
};
static ChunkPlan plan_chunk(const kvpool* p, const LayerState& L, uint32_t first, uint32_t n) {
  ChunkPlan c;
  uint64_t acc = 0;
  for (uint32_t i = 0; i < p->n; ++i) {
    slot_range(*L.map, i, first, n, &c.lo[i], &c.hi[i]);
    c.off[i] = acc;
    if (c.hi[i] == c.lo[i]) continue;
    if (is_hbm(p, i)) { c.hbm_blocks = true; continue; }
    if (is_ssd(p, i)) { c.ssd_blocks = true; continue; }  // through the device's bounce lanes, never through a staging slot
    c.host_blocks = true;
    acc += static_cast<uint64_t>(c.hi[i] - c.lo[i]) * p->payload;
  }
  c.host_bytes = acc;
  return c;
}

// Make `waiter` wait for everything enqueued on `s` so far (a pooled non-timing event; the wait captures the record).
static int stream_after(kvpool* p, cudaStream_t waiter, cudaStream_t s) {
  cudaEvent_t m = nullptr;
  CU(take_event(p, &m));
  CU(cudaEventRecord(m, s));
  CU(cudaStreamWaitEvent(waiter, m, 0));
  p->ev_free.push_back(m);
  return KVPOOL_OK;
}
static void chunk_bases(const kvpool* p, const LayerState& L, const ChunkPlan& c, const StageSlot* slot, LayerArgs* a) {
  for (uint32_t i = 0; i < p->n; ++i) {
    // HBM-type devices: the kernel reaches the stripe in place; host devices: their share of the staging slot
    if (is_hbm(p, i) || !slot) a->pool_base[i] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(p->bufs[i].dev_alias) + L.stripe_off[i]);
    else a->pool_base[i] = reinterpret_cast<uint64_t>(slot->buf) + c.off[i] - static_cast<uint64_t>(c.lo[i]) * p->payload;
  }
}

int kvpool_offload_range(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, uint32_t first_block, uint32_t n_blocks, const void* k_base,
                         const void* v_base, uint64_t stride, const int32_t* table, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
  if (static_cast<uint64_t>(first_block) + n_blocks > L.map->K)
    return fail(KVPOOL_EINVAL, "offload: blocks [%u, %u) exceed the layer's %llu blocks", first_block, first_block + n_blocks,
                (unsigned long long)L.map->K);
  if (L.map->K == 0) { L.offloaded = true; return KVPOOL_OK; }
  if (n_blocks == 0) return KVPOOL_OK;
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const uint32_t N = p->n;
  LayerArgs a = base_args(p, L, k_base, v_base, stride, table_of(pl, layer, table));
  const ChunkPlan whole = plan_chunk(p, L, first_block, n_blocks);
  const bool staged = use_staged(p, true, whole.host_bytes);  // a range is judged by its own size and by where its own blocks sit

  if (!staged) {
    // zero-copy: one kernel gathers the paged blocks and stores them straight into the mapped host stripes
    a.j0 = first_block;
    a.K = n_blocks;
    if (n_blocks == L.map->K) a.visit = L.map->visit_d;  // (null unless the pool mixes host and HBM-type devices)
    chunk_bases(p, L, ChunkPlan{}, nullptr, &a);
    if (L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));  // an earlier staged offload of this layer still in flight
    rc = launch_counted(p, a, true, true, s);
    if (rc != KVPOOL_OK) return rc;
    mark_offloaded(L, first_block, n_blocks);  // only now: a failed launch must not leave the blocks flagged as present
    CU(cudaEventRecord(L.landed, s));
    L.landed_pending = true;
    return note_use(p, pl, s);
  }

  // staged: pack kernel -> device staging slot, then one D2H copy per device on the per-device I/O streams; `stream` is
  // released as soon as the last pack is enqueued.  A layer larger than a slot travels in chunks of logical blocks.
  const uint64_t per_slot = p->slots.empty() ? 0 : blocks_per_slot(p);
  if (per_slot == 0 && whole.host_blocks) return fail(KVPOOL_ESTATE, "offload: no staging slot (the placement was made while the path was zero-copy)");
  // `landed` must mean "all stripes complete": it is recorded on a stream of the pool's own that carries no copies and only
  // gathers every chunk's kernel and copies — the per-device I/O streams never wait for one another
  cudaStream_t lead = p->join_out;
  if (L.landed_pending) CU(cudaStreamWaitEvent(lead, L.landed, 0));  // `landed` keeps covering what was offloaded before
  // an earlier offload of this layer may still be writing the HBM-type stripes the kernel stores into
  if (whole.hbm_blocks && L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
  if (n_blocks > per_slot || p->ssd_mask) {
    // DEVICE-MAJOR chunks: a chunk is a run of consecutive slots of one device's stripe, gathered by a launch that finds its
    // logical blocks through that device's inverse map, and leaves the slot as ONE copy.  An HBM-type device's share is
    // gathered in place by one launch; an SSD-type device's share goes through that device's bounce lanes (SSD_Direct_Store,
    // Alg. 1 l.20-21), which is why a pool with such a device always moves device-major.
    a.order = L.map->order_d;
    for (uint32_t i = 0; i < N; ++i) {
      if (is_ssd(p, i)) {
        if (whole.hi[i] > whole.lo[i] && (rc = ssd_move(p, L, i, whole.lo[i], whole.hi[i], true, a, s)) != KVPOOL_OK) return rc;
        continue;
      }
      for (uint32_t lo = whole.lo[i]; lo < whole.hi[i];) {
        const uint32_t n = is_hbm(p, i) ? whole.hi[i] - lo : static_cast<uint32_t>(std::min<uint64_t>(per_slot, whole.hi[i] - lo));
        a.j0 = L.map->start[i] + lo;
        a.K = n;
        uint8_t* const stripe_at = static_cast<uint8_t*>(p->bufs[i].dev_alias) + L.stripe_off[i] + static_cast<uint64_t>(lo) * p->payload;
        lo += n;
        if (is_hbm(p, i)) {
          a.pool_base[0] = reinterpret_cast<uint64_t>(stripe_at);
          rc = launch_counted(p, a, true, false, s);
          if (rc != KVPOOL_OK) return rc;
          continue;
        }
        StageSlot& slot = p->slots[p->slot_cursor++ % p->slots.size()];
        rc = wait_slot_free(p, slot, s);
        if (rc != KVPOOL_OK) return rc;
        slot.copies_after_kernel = 0;
        a.pool_base[0] = reinterpret_cast<uint64_t>(slot.buf);
        rc = launch_counted(p, a, true, false, s);
        if (rc != KVPOOL_OK) return rc;
        CU(cudaEventRecord(slot.kernel_done, s));
        CU(cudaStreamWaitEvent(p->io_out[i], slot.kernel_done, 0));
        if (L.landed_pending) CU(cudaStreamWaitEvent(p->io_out[i], L.landed, 0));  // the previous offload of this layer
        CU(cudaMemcpyAsync(static_cast<uint8_t*>(p->bufs[i].host) + (stripe_at - static_cast<uint8_t*>(p->bufs[i].dev_alias)), slot.buf,
                           static_cast<uint64_t>(n) * p->payload, cudaMemcpyDeviceToHost, p->io_out[i]));
        p->n_memcpys++;
        CU(cudaEventRecord(slot.copy_done[i], p->io_out[i]));
        slot.copies_after_kernel = 1u << i;
        CU(cudaStreamWaitEvent(lead, slot.copy_done[i], 0));
      }
    }
  } else {
    const ChunkPlan& c = whole;  // the range fits one staging slot: one pack launch, one copy per device
    a.j0 = first_block;
    a.K = n_blocks;
    if (!c.host_blocks) {  // the whole range sits on HBM-type devices: nothing to stage, no slot taken
      chunk_bases(p, L, c, nullptr, &a);
      rc = launch_counted(p, a, true, false, s);
      if (rc != KVPOOL_OK) return rc;
    } else {
      StageSlot& slot = p->slots[p->slot_cursor++ % p->slots.size()];
      rc = wait_slot_free(p, slot, s);
      if (rc != KVPOOL_OK) return rc;
      slot.copies_after_kernel = 0;
      chunk_bases(p, L, c, &slot, &a);
      rc = launch_counted(p, a, true, false, s);
      if (rc != KVPOOL_OK) return rc;
      CU(cudaEventRecord(slot.kernel_done, s));
      for (uint32_t i = 0; i < N; ++i) {
        if (c.hi[i] == c.lo[i] || is_hbm(p, i)) continue;
        const uint64_t bytes = static_cast<uint64_t>(c.hi[i] - c.lo[i]) * p->payload;
        CU(cudaStreamWaitEvent(p->io_out[i], slot.kernel_done, 0));
        if (L.landed_pending) CU(cudaStreamWaitEvent(p->io_out[i], L.landed, 0));  // the previous offload of this layer
        CU(cudaMemcpyAsync(static_cast<uint8_t*>(p->bufs[i].host) + L.stripe_off[i] + static_cast<uint64_t>(c.lo[i]) * p->payload,
                           slot.buf + c.off[i], bytes, cudaMemcpyDeviceToHost, p->io_out[i]));
        p->n_memcpys++;
        CU(cudaEventRecord(slot.copy_done[i], p->io_out[i]));
        slot.copies_after_kernel |= 1u << i;
      }
      for (uint32_t i = 0; i < N; ++i)
        if (slot.copies_after_kernel >> i & 1u) CU(cudaStreamWaitEvent(lead, slot.copy_done[i], 0));
    }
  }
  if (whole.hbm_blocks) {  // `landed` also covers the HBM-type stripes the kernels on `s` wrote in place
    rc = stream_after(p, lead, s);
    if (rc != KVPOOL_OK) return rc;
  }
  mark_offloaded(L, first_block, n_blocks);  // every chunk is enqueued (an error above leaves the range unflagged: retrieve -> ESTATE)
  CU(cudaEventRecord(L.landed, lead));
  L.landed_pending = true;
  return note_use(p, pl, s);
}

int kvpool_offload(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, const void* k_base, const void* v_base, uint64_t stride,
                   const int32_t* table, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "offload: bad pool or placement");
  if (layer >= p->geom.n_layers) return fail(KVPOOL_EINVAL, "layer %u out of range (n_layers %u)", layer, p->geom.n_layers);
  return kvpool_offload_range(p, pl, layer, 0, static_cast<uint32_t>(pl->layers[layer].map->K), k_base, v_base, stride, table, cuda_stream);
}

int kvpool_retrieve_range(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, uint32_t first_block, uint32_t n_blocks, void* k_base,
                          void* v_base, uint64_t stride, const int32_t* table, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
  if (static_cast<uint64_t>(first_block) + n_blocks > L.map->K)
    return fail(KVPOOL_EINVAL, "retrieve: blocks [%u, %u) exceed the layer's %llu blocks", first_block, first_block + n_blocks,
                (unsigned long long)L.map->K);
  if (!L.offloaded && L.have.empty()) return fail(KVPOOL_ESTATE, "retrieve: layer %u was never offloaded", layer);
  if (!is_offloaded(L, first_block, n_blocks))
    return fail(KVPOOL_ESTATE, "retrieve: some of blocks [%u, %u) of layer %u were never offloaded", first_block, first_block + n_blocks, layer);
  if (n_blocks == 0) return KVPOOL_OK;
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const uint32_t N = p->n;
  LayerArgs a = base_args(p, L, k_base, v_base, stride, table_of(pl, layer, table));
  const ChunkPlan whole = plan_chunk(p, L, first_block, n_blocks);
  // staged only if something travels through the copy engines (a range whose blocks all sit on HBM-type devices has
  // nothing to stage) and, on the auto path, enough of it
  const bool staged = use_staged(p, false, whole.host_bytes);
  settle_landed(L);

  if (!staged) {
    a.j0 = first_block;
    a.K = n_blocks;
    if (n_blocks == L.map->K) a.visit = L.map->visit_d;
    chunk_bases(p, L, ChunkPlan{}, nullptr, &a);
    if (L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
    rc = launch_counted(p, a, false, true, s);
    return rc == KVPOOL_OK ? note_use(p, pl, s) : rc;
  }

  // staged: one H2D copy per device (only the slots the range touches) on the per-device I/O streams — these may run
  // ahead of `stream` — then the unpack kernel on `stream` once all of them have landed in the staging slot.  A range
  // larger than a slot travels in chunks of logical blocks: the copies of chunk c+1 overlap the unpack of chunk c.
  const uint64_t per_slot = p->slots.empty() ? 0 : blocks_per_slot(p);
  if (per_slot == 0 && whole.host_blocks) return fail(KVPOOL_ESTATE, "retrieve: no staging slot (the placement was made while the path was zero-copy)");
  if (whole.hbm_blocks && L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));  // HBM-type stripes are read in place
  if (n_blocks > per_slot || p->ssd_mask) {
    // DEVICE-MAJOR chunks (see kvpool_offload_range): one copy fills a slot with a run of one device's slots, one launch
    // scatters them through that device's inverse map; the copy of the next chunk overlaps it.  SSD-type devices first: their
    // retrieve commands (SSD_Direct_Retrieve) go to the workers before anything is enqueued for the faster
    // devices, so that the disks read while the link moves the host-memory devices' share.
    a.order = L.map->order_d;
    for (uint32_t i = 0; i < N; ++i)
      if (is_ssd(p, i) && whole.hi[i] > whole.lo[i] && (rc = ssd_move(p, L, i, whole.lo[i], whole.hi[i], false, a, s)) != KVPOOL_OK) return rc;
    for (uint32_t i = 0; i < N; ++i) {
      if (is_ssd(p, i)) continue;
      for (uint32_t lo = whole.lo[i]; lo < whole.hi[i];) {
        const uint32_t n = is_hbm(p, i) ? whole.hi[i] - lo : static_cast<uint32_t>(std::min<uint64_t>(per_slot, whole.hi[i] - lo));
        a.j0 = L.map->start[i] + lo;
        a.K = n;
        const uint64_t at = L.stripe_off[i] + static_cast<uint64_t>(lo) * p->payload;
        lo += n;
        if (is_hbm(p, i)) {
          a.pool_base[0] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(p->bufs[i].dev_alias) + at);
          rc = launch_counted(p, a, false, false, s);
          if (rc != KVPOOL_OK) return rc;
          continue;
        }
        StageSlot& slot = p->slots[p->slot_cursor++ % p->slots.size()];
        rc = wait_slot_free(p, slot, p->io[i]);
        if (rc != KVPOOL_OK) return rc;
        if (L.landed_pending) CU(cudaStreamWaitEvent(p->io[i], L.landed, 0));
        slot.copies_after_kernel = 0;
        CU(cudaMemcpyAsync(slot.buf, static_cast<uint8_t*>(p->bufs[i].host) + at, static_cast<uint64_t>(n) * p->payload, cudaMemcpyHostToDevice, p->io[i]));
        p->n_memcpys++;
        CU(cudaEventRecord(slot.copy_done[i], p->io[i]));
        CU(cudaStreamWaitEvent(s, slot.copy_done[i], 0));
        a.pool_base[0] = reinterpret_cast<uint64_t>(slot.buf);
        rc = launch_counted(p, a, false, false, s);
        if (rc != KVPOOL_OK) return rc;
        CU(cudaEventRecord(slot.kernel_done, s));
      }
    }
    return note_use(p, pl, s);
  }
  {
    const ChunkPlan& c = whole;  // the range fits one staging slot: one copy per device, one unpack launch
    a.j0 = first_block;
    a.K = n_blocks;
    StageSlot& slot = p->slots[p->slot_cursor++ % p->slots.size()];
    for (uint32_t i = 0; i < N; ++i) {
      if (c.hi[i] == c.lo[i] || is_hbm(p, i)) continue;
      rc = wait_slot_free(p, slot, p->io[i]);
      if (rc != KVPOOL_OK) return rc;
      if (L.landed_pending) CU(cudaStreamWaitEvent(p->io[i], L.landed, 0));
    }
    slot.copies_after_kernel = 0;
    chunk_bases(p, L, c, &slot, &a);
    for (uint32_t i = 0; i < N; ++i) {
      if (c.hi[i] == c.lo[i] || is_hbm(p, i)) continue;
      const uint64_t bytes = static_cast<uint64_t>(c.hi[i] - c.lo[i]) * p->payload;
      CU(cudaMemcpyAsync(slot.buf + c.off[i], static_cast<uint8_t*>(p->bufs[i].host) + L.stripe_off[i] + static_cast<uint64_t>(c.lo[i]) * p->payload,
                         bytes, cudaMemcpyHostToDevice, p->io[i]));
      p->n_memcpys++;
      CU(cudaEventRecord(slot.copy_done[i], p->io[i]));
      CU(cudaStreamWaitEvent(s, slot.copy_done[i], 0));
    }
    rc = launch_counted(p, a, false, false, s);
    if (rc != KVPOOL_OK) return rc;
    CU(cudaEventRecord(slot.kernel_done, s));
  }
  return note_use(p, pl, s);
}


int kvpool_retrieve(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, void* k_base, void* v_base, uint64_t stride,
                    const int32_t* table, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "retrieve: bad pool or placement");
  if (layer >= p->geom.n_layers) return fail(KVPOOL_EINVAL, "layer %u out of range (n_layers %u)", layer, p->geom.n_layers);
  return kvpool_retrieve_range(p, pl, layer, 0, static_cast<uint32_t>(pl->layers[layer].map->K), k_base, v_base, stride, table, cuda_stream);
}

namespace {
struct LayerGroup {  // a run of layers of one batched call that moves as one unit
  uint32_t q[kMaxBatch];  // indices into the call's pointer arrays (layer = first + q)
  uint32_t n = 0;
  uint64_t bytes = 0;
  uint64_t host_bytes = 0;  // of which on host-memory devices (what the staged path would send through the copy engines)
};
struct BatchCall {
  kvpool* p;
  kvpool_placement* pl;
  bool pack;
  uint32_t first;
  const void* const* k_bases;
  const void* const* v_bases;
  const int32_t* const* tables;
  uint64_t stride;
  cudaStream_t s;
  void* const* ready;  // optional: caller-owned cudaEvent_t per layer of the call, recorded on `s` when that layer is complete
  bool* chain_run;     // the launch enqueued last on `s` by this call heads / follows a run of chained launches (kernels.cuh)
  std::vector<LayerState*>* landed_later;  // offloads of a chained run: their `landed` events are recorded behind the run
  bool signal;         // a small request with a consumer behind per-layer events: groups move zero-copy, ONE launch that
                       // raises a flag per layer (kernels.cuh); *signalled says the group's ready events are taken care of
  bool* signalled;
};

// The next set of per-layer flags (round-robin over kSignalSets, made on first use); `s` waits for the launch that used it last.
int take_signal_set(kvpool* p, cudaStream_t s, SignalSet** out) {
  if (p->sig.empty()) {
    std::vector<SignalSet> v(kSignalSets);
    for (auto& x : v) {
      CU(cudaMalloc(reinterpret_cast<void**>(&x.mem_d), 2ull * kMaxBatch * sizeof(uint32_t)));
      CU(cudaMemsetAsync(x.mem_d, 0, 2ull * kMaxBatch * sizeof(uint32_t), p->upload));
      CU(cudaStreamCreateWithFlags(&x.stream, cudaStreamNonBlocking));
      CU(cudaEventCreateWithFlags(&x.done, cudaEventDisableTiming));
      p->own_streams.push_back(x.stream);  // kvpool_release / kvpool_synchronize wait for them too
    }
    CU(cudaStreamSynchronize(p->upload));
    p->sig = std::move(v);
  }
  SignalSet& x = p->sig[p->sig_cursor++ % p->sig.size()];
  CU(cudaStreamWaitEvent(s, x.done, 0));
  *out = &x;
  return KVPOOL_OK;
}

// Record the `landed` events a chained run of offload launches has put off (an event record between two launches would
// undo the chaining): behind the run's last launch every one of its layers is complete in the pool.
int flush_landed(const BatchCall& c) {
  for (LayerState* L : *c.landed_later) {
    CU(cudaEventRecord(L->landed, c.s));
    L->landed_pending = true;
  }
  c.landed_later->clear();
  return KVPOOL_OK;
}

void fill_descs(const BatchCall& c, const LayerGroup& g, MultiArgs* ma) {
  ma->stride = c.stride;
  ma->kvb = static_cast<uint32_t>(c.p->kvb);
  ma->nphys_check = c.p->check_nphys;
  ma->bad = c.p->bad_d;
  ma->n = g.n;
  ma->total_units = 0;
  for (uint32_t b = 0; b < g.n; ++b) {
    const LayerState& L = c.pl->layers[c.first + g.q[b]];
    MultiDesc& d = ma->d[b];
    d.k_base = static_cast<uint8_t*>(const_cast<void*>(c.k_bases[g.q[b]]));
    d.v_base = static_cast<uint8_t*>(const_cast<void*>(c.v_bases[g.q[b]]));
    d.table = table_of(c.pl, c.first + g.q[b], c.tables ? c.tables[g.q[b]] : nullptr);
    d.dev = L.map->dev_d;
    d.slot = L.map->slot_d;
    d.pool_base = L.base_d;
    d.K = static_cast<uint32_t>(L.map->K);
    d.first_unit = ma->total_units;
    ma->total_units += d.K;
  }
}

// Zero-copy: one kernel moves the whole group straight between the paged blocks and the mapped host stripes.
int issue_zero_copy_group(const BatchCall& c, const LayerGroup& g) {
  kvpool* p = c.p;
  MultiArgs ma{};
  fill_descs(c, g, &ma);
  bool waited = false;
  for (uint32_t b = 0; b < g.n; ++b) {
    LayerState& L = c.pl->layers[c.first + g.q[b]];
    if (L.landed_pending) { CU(cudaStreamWaitEvent(c.s, L.landed, 0)); waited = true; }  // settled (no wait) after kvpool_synchronize
  }
  // Retrieves of one batched call in a pool with HBM-type devices: the launches are independent of each other (other
  // stripes, other paged tensors) and last ~90 us each, of which the first microseconds are the link's first-byte latency
  // and the ramp: chain them (kernels.cuh), so that a launch's host-memory blocks are already on the link while its
  // predecessor's last wave drains.  Only where the launches are back to back on the stream (no event wait or record
  // between them, no profiling markers) and many waves long (the HBM grid; a 4-CTA link launch would let the whole
  // request start at once and lose the layer order).
  if (c.signal && !c.pack && g.n > 1) {
    // ONE launch for the group, and still one hand-over per layer: the kernel raises a flag when a layer's last piece has
    // landed; a stream of the flag set's own waits for the flags in layer order and records the caller's events behind them
    SignalSet* x = nullptr;
    int rc = take_signal_set(p, c.s, &x);
    if (rc != KVPOOL_OK) return rc;
    ma.sig_count = x->mem_d;
    ma.sig_flag = x->mem_d + kMaxBatch;
    ma.sig_seq = ++x->seq;
    *c.chain_run = false;
    if ((rc = flush_landed(c)) != KVPOOL_OK) return rc;
    if ((rc = launch_multi_counted(p, ma, false, true, c.s)) != KVPOOL_OK) return rc;
    CU(cudaEventRecord(x->done, c.s));
    for (uint32_t b = 0; b < g.n; ++b) {
      if (!c.ready[g.q[b]]) continue;
      if ((rc = stream_wait_geq(x->stream, reinterpret_cast<uint64_t>(ma.sig_flag + b), ma.sig_seq)) != KVPOOL_OK) return rc;
      CU(cudaEventRecord(static_cast<cudaEvent_t>(c.ready[g.q[b]]), x->stream));
    }
    *c.signalled = true;
    return KVPOOL_OK;
  }
  const bool chain = p->hbm_mask && !c.ready && !waited && !p->profiling && p->tune.pdl != 2;
  ma.chain = !chain ? kChainNone : (*c.chain_run ? kChainFollower : kChainHead);
  if (!chain) {
    const int frc = flush_landed(c);
    if (frc != KVPOOL_OK) return frc;
  }
  *c.chain_run = chain;
  const int rc = launch_multi_counted(p, ma, c.pack, true, c.s);
  if (rc != KVPOOL_OK) return rc;
  if (c.pack)
    for (uint32_t b = 0; b < g.n; ++b) {
      LayerState& L = c.pl->layers[c.first + g.q[b]];
      L.offloaded = true;
      L.have.clear();
      if (chain) { c.landed_later->push_back(&L); continue; }
      CU(cudaEventRecord(L.landed, c.s));
      L.landed_pending = true;
    }
  return KVPOOL_OK;
}

// Staged: the group's stripes are one contiguous span per pool device (region allocation in kvpool_place), so the
// whole group moves with ONE cudaMemcpyAsync per device and ONE pack / unpack launch.  Returns 1 if the group does
// not fit a staging slot (the caller then falls back to per-layer calls).
int issue_staged_group(const BatchCall& c, const LayerGroup& g) {
  kvpool* p = c.p;
  *c.chain_run = false;
  if (const int frc = flush_landed(c)) return frc;
  if (p->ssd_mask) return 1;  // a pool with an SSD-type device moves layer by layer, device-major
  const uint32_t N = p->n;
  const std::vector<cudaStream_t>& ios = c.pack ? p->io_out : p->io;  // the copy streams of this direction
  const LayerState& A = c.pl->layers[c.first + g.q[0]];
  const LayerState& Z = c.pl->layers[c.first + g.q[g.n - 1]];
  // span[i]: bytes device i's copy engine moves for the group.  HBM-type devices move nothing that way — the kernel
  // reaches their stripes in place (delta 0) — so they take no room in the staging slot either.
  uint64_t span_lo[KVPOOL_MAX_DEVICES], span[KVPOOL_MAX_DEVICES], dev_start[KVPOOL_MAX_DEVICES], total = 0;
  bool hbm_blocks = false;
  for (uint32_t i = 0; i < N; ++i) {
    span_lo[i] = A.stripe_off[i];
    span[i] = Z.stripe_off[i] + static_cast<uint64_t>(Z.map->counts[i]) * p->payload - span_lo[i];
    if (is_hbm(p, i)) { hbm_blocks |= span[i] != 0; span[i] = 0; }
    dev_start[i] = total;
    total += (span[i] + 255) / 256 * 256;
  }
  if (p->slots.empty() || total > p->slot_bytes || (p->tune.stage_chunk_bytes && total > std::max<uint64_t>(p->tune.stage_chunk_bytes, p->payload) + 256ull * N))
    return 1;
  if (total == 0) return issue_zero_copy_group(c, g);  // every block of the group sits on HBM-type devices: nothing to stage, no slot taken
  StageSlot& slot = p->slots[p->slot_cursor++ % p->slots.size()];
  MultiArgs ma{};
  fill_descs(c, g, &ma);
  for (uint32_t i = 0; i < N; ++i)
    ma.delta[i] = is_hbm(p, i) ? 0
                               : reinterpret_cast<uint64_t>(slot.buf + dev_start[i]) - reinterpret_cast<uint64_t>(static_cast<uint8_t*>(p->bufs[i].dev_alias) + span_lo[i]);

  // an earlier offload of these layers that is still in flight must land before their stripes are touched again:
  // gather those waits on the first I/O stream that has work and fan out through one event; the kernel's own stream
  // waits too when it touches HBM-type stripes directly
  cudaStream_t lead = nullptr;
  for (uint32_t i = 0; i < N && !lead; ++i)
    if (span[i]) lead = ios[i];
  bool gated = false;
  for (uint32_t b = 0; b < g.n; ++b) {
    LayerState& L = c.pl->layers[c.first + g.q[b]];
    settle_landed(L);
    if (!L.landed_pending) continue;
    if (lead) { CU(cudaStreamWaitEvent(lead, L.landed, 0)); gated = true; }
    if (hbm_blocks) CU(cudaStreamWaitEvent(c.s, L.landed, 0));
  }

  int rc;
  if (c.pack) {
    rc = wait_slot_free(p, slot, c.s);
    if (rc != KVPOOL_OK) return rc;
    slot.copies_after_kernel = 0;
    rc = launch_multi_counted(p, ma, true, false, c.s);
    if (rc != KVPOOL_OK) return rc;
    CU(cudaEventRecord(slot.kernel_done, c.s));
    if (gated) CU(cudaEventRecord(slot.gate, lead));
    for (uint32_t i = 0; i < N; ++i) {
      if (!span[i]) continue;
      CU(cudaStreamWaitEvent(ios[i], slot.kernel_done, 0));
      if (gated && ios[i] != lead) CU(cudaStreamWaitEvent(ios[i], slot.gate, 0));
      CU(cudaMemcpyAsync(static_cast<uint8_t*>(p->bufs[i].host) + span_lo[i], slot.buf + dev_start[i], span[i], cudaMemcpyDeviceToHost, ios[i]));
      p->n_memcpys++;
      CU(cudaEventRecord(slot.copy_done[i], ios[i]));
      slot.copies_after_kernel |= 1u << i;
    }
    for (uint32_t i = 0; i < N; ++i)
      if (span[i] && ios[i] != lead) CU(cudaStreamWaitEvent(lead, slot.copy_done[i], 0));
    for (uint32_t b = 0; b < g.n; ++b) {  // `lead` has waited for the kernel and every copy; with no host stripe the kernel was all
      LayerState& L = c.pl->layers[c.first + g.q[b]];
      L.offloaded = true;
      L.have.clear();
      CU(cudaEventRecord(L.landed, lead ? lead : c.s));
      L.landed_pending = true;
    }
    return KVPOOL_OK;
  }
  for (uint32_t i = 0; i < N; ++i) {
    if (!span[i]) continue;
    rc = wait_slot_free(p, slot, ios[i]);
    if (rc != KVPOOL_OK) return rc;
  }
  slot.copies_after_kernel = 0;
  if (gated) CU(cudaEventRecord(slot.gate, lead));
  for (uint32_t i = 0; i < N; ++i) {
    if (!span[i]) continue;
    if (gated && ios[i] != lead) CU(cudaStreamWaitEvent(ios[i], slot.gate, 0));
    CU(cudaMemcpyAsync(slot.buf + dev_start[i], static_cast<uint8_t*>(p->bufs[i].host) + span_lo[i], span[i], cudaMemcpyHostToDevice, ios[i]));
    p->n_memcpys++;
    CU(cudaEventRecord(slot.copy_done[i], ios[i]));
    CU(cudaStreamWaitEvent(c.s, slot.copy_done[i], 0));
  }
  rc = launch_multi_counted(p, ma, false, false, c.s);
  if (rc != KVPOOL_OK) return rc;
  CU(cudaEventRecord(slot.kernel_done, c.s));
  return KVPOOL_OK;
}

int issue_group_work(const BatchCall& c, const LayerGroup& g);

// Move one group, then tell the caller's per-layer events: the layers of a group become ready together.
int issue_group(const BatchCall& c, const LayerGroup& g) {
  if (g.n == 0) return KVPOOL_OK;
  *c.signalled = false;
  const int rc = issue_group_work(c, g);
  if (rc != KVPOOL_OK || !c.ready || *c.signalled) return rc;
  for (uint32_t b = 0; b < g.n; ++b)
    if (c.ready[g.q[b]]) CU(cudaEventRecord(static_cast<cudaEvent_t>(c.ready[g.q[b]]), c.s));
  return KVPOOL_OK;
}

int issue_group_work(const BatchCall& c, const LayerGroup& g) {
  kvpool* p = c.p;
  if ((c.signal && !p->ssd_mask) || !use_staged(p, c.pack, g.host_bytes)) return issue_zero_copy_group(c, g);
  if (g.n > 1) {
    const int rc = issue_staged_group(c, g);
    if (rc != 1) return rc;
  }
  *c.chain_run = false;
  if (const int frc = flush_landed(c)) return frc;
  for (uint32_t b = 0; b < g.n; ++b) {  // a single layer, or a group too large for a staging slot: the per-layer path
    const uint32_t q = g.q[b], layer = c.first + q;
    const int rc = c.pack ? kvpool_offload(p, c.pl, layer, c.k_bases[q], c.v_bases[q], c.stride, c.tables ? c.tables[q] : nullptr, c.s)
                          : kvpool_retrieve(p, c.pl, layer, const_cast<void*>(c.k_bases[q]), const_cast<void*>(c.v_bases[q]), c.stride, c.tables ? c.tables[q] : nullptr, c.s);
    if (rc != KVPOOL_OK) return rc;
  }
  return KVPOOL_OK;
}
}  // namespace

// Layers [first, first+n) in one call.  Consecutive layers are gathered into groups of at least tune.group_bytes (a
// layer at least that large travels with whatever small layers precede it); each group moves as one unit: one fused
// zero-copy launch, or one pack/unpack launch plus one copy per pool device.
static int layers_batched_locked(kvpool_t* p, kvpool_placement_t* pl, bool pack, uint32_t first, uint32_t n, const void* const* k_bases,
                                 const void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream,
                                 void* const* ready);

static int layers_batched(kvpool_t* p, kvpool_placement_t* pl, bool pack, uint32_t first, uint32_t n, const void* const* k_bases,
                          const void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream,
                          void* const* ready = nullptr) {
  PoolLock lock__(p);
  if (!p || !pack || !p->ssd_mask) return layers_batched_locked(p, pl, pack, first, n, k_bases, v_bases, stride, tables, cuda_stream, ready);
  // a batched offload over a pool with SSD-type devices: their pack launches (kvpool_ssd.cu) are joined back to `stream`
  // once, here, instead of after every layer, so that the launches of the host-memory devices never queue behind a disk
  p->ssd_defer_join = true;
  int rc = layers_batched_locked(p, pl, pack, first, n, k_bases, v_bases, stride, tables, cuda_stream, ready);
  p->ssd_defer_join = false;
  DeviceGuard guard(p->cuda_device);
  const int rc2 = ssd_join_deferred(p, static_cast<cudaStream_t>(cuda_stream));  // (also after an error: the launches made so far still read the source)
  if (rc == KVPOOL_OK) rc = rc2;
  if (rc == KVPOOL_OK && pl) rc = note_use(p, pl, static_cast<cudaStream_t>(cuda_stream));
  return rc;
}

static int layers_batched_locked(kvpool_t* p, kvpool_placement_t* pl, bool pack, uint32_t first, uint32_t n, const void* const* k_bases,
                                 const void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream,
                                 void* const* ready) {
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "layers: bad pool or placement");
  if (static_cast<uint64_t>(first) + n > p->geom.n_layers) return fail(KVPOOL_EINVAL, "layers [%u, %u) out of range (n_layers %u)", first, first + n, p->geom.n_layers);
  if (n == 0) return KVPOOL_OK;
  if (!k_bases || !v_bases) return fail(KVPOOL_EINVAL, "layers: null pointer array");
  if (!tables && !pl->own_tables_set) return fail(KVPOOL_EINVAL, "layers: null block_tables (and no tables uploaded with kvpool_set_tables)");
  for (uint32_t q = 0; q < n; ++q) {  // validate everything first: no partial effects on EINVAL / ESTATE
    const int rc = check_layer_call(p, pl, first + q, k_bases[q], v_bases[q], stride, tables ? tables[q] : nullptr);
    if (rc != KVPOOL_OK) return rc;
    if (!pack && !pl->layers[first + q].offloaded) return fail(KVPOOL_ESTATE, "retrieve: layer %u was never offloaded", first + q);
  }
  DeviceGuard guard(p->cuda_device);
  bool chain_run = false;
  std::vector<LayerState*> landed_later;
  uint64_t cap = std::max<uint64_t>(p->tune.group_bytes, 1);
  bool signal = false, signalled = false;
  uint64_t tail_start = ~0ull;  // bytes of the call in front of its last, short group (below)
  if (ready) {
    // A consumer follows behind the per-layer events.  On the zero-copy path a request so small that it would travel as
    // one or two groups (all of a group's layers ready together: the consumer hardly overlapped) moves as ONE launch that
    // signals every layer as it completes, so that the consumer of layer l runs under the transfer of layer l+1.  (Not
    // the default for such requests: through the copy engines the link runs 8 % faster than under SM-issued reads, and two
    // staged groups beat the signalled launch — GPT-OSS-shaped KV at 1K context, 27 MiB: 0.566 against 0.594 ms.)
    uint64_t total = 0;
    for (uint32_t q = 0; q < n; ++q) total += pl->layers[first + q].map->K * p->payload;
    if (!pack && total < 2 * cap && p->path == KVPOOL_PATH_ZEROCOPY && !p->ssd_mask && memops_init() == KVPOOL_OK) {
      signal = true;
      cap = std::max<uint64_t>(total, 1);
    } else if (total < cap) {
      cap = std::max<uint64_t>((total + 1) / 2, 1);  // else cut it in two, so that the first half's consumer runs under the second half's transfer
    }
    // ... and whatever the size: the layers of the call's LAST group become ready together when the last byte has arrived,
    // and their consumers then run with nothing left to hide under (a dozen small launches: 40-60 us behind a 0.5-2.5 ms
    // request).  So the last eighth of a small request (at most a quarter of a group) travels as a short group of its own:
    // one more set of copies (~10 us of ramps) for a tail of two or three consumers instead of twelve or sixteen.
    if (!signal) tail_start = total - std::min(total / 8, cap / 4);
  }
  const BatchCall c{p, pl, pack, first, k_bases, v_bases, tables, stride, static_cast<cudaStream_t>(cuda_stream), ready, &chain_run, &landed_later,
                    signal, &signalled};
  struct Flush {  // whatever path leaves the call: the events put off so far are recorded
    const BatchCall& c;
    ~Flush() { flush_landed(c); }
  } flush_on_exit{c};
  LayerGroup g;
  uint64_t units = 0, before = 0;  // before: bytes of the call's layers in front of layer q
  bool tail_open = false;
  for (uint32_t q = 0; q < n; ++q) {
    LayerState& L = pl->layers[first + q];
    if (L.map->K == 0) {  // nothing to move: ready in stream order right away
      if (pack) L.offloaded = true;
      if (ready && ready[q]) CU(cudaEventRecord(static_cast<cudaEvent_t>(ready[q]), c.s));
      continue;
    }
    const uint64_t bytes = L.map->K * p->payload;
    if (!tail_open && before >= tail_start) {  // the short last group starts here
      tail_open = true;
      if (g.n) {
        const int rc = issue_group(c, g);
        if (rc != KVPOOL_OK) return rc;
        g = LayerGroup{};
        units = 0;
      }
    }
    before += bytes;
    if (g.n && (g.n == kMaxBatch || units + L.map->K > 0x7fffffffull || g.bytes + bytes > std::max(cap, bytes))) {
      const int rc = issue_group(c, g);
      if (rc != KVPOOL_OK) return rc;
      g = LayerGroup{};
      units = 0;
    }
    g.q[g.n++] = q;
    g.bytes += bytes;
    g.host_bytes += L.map->host_blocks * p->payload;
    units += L.map->K;
    if (g.bytes >= cap) {  // on every path: a group is also the grain at which a consumer's per-layer events fire
      const int rc = issue_group(c, g);
      if (rc != KVPOOL_OK) return rc;
      g = LayerGroup{};
      units = 0;
    }
  }
  int rc = issue_group(c, g);
  if (rc == KVPOOL_OK) rc = flush_landed(c);
  return rc == KVPOOL_OK ? note_use(p, pl, c.s) : rc;
}

int kvpool_offload_layers(kvpool_t* p, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers, const void* const* k_bases,
                          const void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream) {
  return layers_batched(p, pl, true, first_layer, n_layers, k_bases, v_bases, stride, tables, cuda_stream);
}

int kvpool_retrieve_layers(kvpool_t* p, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers, void* const* k_bases,
                           void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream) {
  return layers_batched(p, pl, false, first_layer, n_layers, k_bases, v_bases, stride, tables, cuda_stream);
}

int kvpool_retrieve_layers_signal(kvpool_t* p, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers, void* const* k_bases,
                                  void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* const* layer_ready,
                                  void* cuda_stream) {
  if (n_layers && !layer_ready) return fail(KVPOOL_EINVAL, "retrieve_layers_signal: null layer_ready array");
  return layers_batched(p, pl, false, first_layer, n_layers, k_bases, v_bases, stride, tables, cuda_stream, layer_ready);
}

int kvpool_set_tables(kvpool_t* p, kvpool_placement_t* pl, const int32_t* tables_host, uint64_t n_entries, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "set_tables: bad pool or placement");
  uint64_t total = 0;
  for (auto& L : pl->layers) total += L.map->K;
  if (n_entries != total) return fail(KVPOOL_EINVAL, "set_tables: %llu entries given, the placement's layers hold %llu blocks", (unsigned long long)n_entries, (unsigned long long)total);
  if (total == 0) { pl->own_tables_set = true; pl->own_table_off.assign(pl->layers.size(), 0); return KVPOOL_OK; }
  if (!tables_host) return fail(KVPOOL_EINVAL, "set_tables: null tables_host");
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (!pl->own_tables_d) {
    const uint64_t bytes = (total * 4 + 255) / 256 * 256;
    uint64_t off = 0;
    if (p->table_alloc.alloc(bytes, &off)) {
      pl->own_tables_d = reinterpret_cast<int32_t*>(p->table_arena + off);
      pl->own_tables_in_arena = true;
    } else {
      cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&pl->own_tables_d), bytes);
      if (e != cudaSuccess) { cudaGetLastError(); pl->own_tables_d = nullptr; return fail(KVPOOL_ENOMEM, "set_tables: %s", cudaGetErrorString(e)); }
      pl->own_tables_in_arena = false;
    }
    pl->own_tables_bytes = bytes;
    pl->own_table_off.resize(pl->layers.size());
    uint64_t acc = 0;
    for (size_t l = 0; l < pl->layers.size(); ++l) { pl->own_table_off[l] = acc; acc += pl->layers[l].map->K; }
  }
  if (pl->own_tables_in_arena) {
    // through the pinned mirror of the arena: the caller's buffer (pageable or not) is free again when the call returns,
    // and the copy is one asynchronous DMA ordered on `stream`.  A re-upload first waits for the work enqueued with the
    // placement so far (the earlier upload may not have read the mirror yet; kernels may still read the old tables).
    if (pl->own_tables_set)
      for (auto& u : pl->last_use) CU(cudaEventSynchronize(u.second));
    uint8_t* mirror = p->table_arena_host + (reinterpret_cast<uint8_t*>(pl->own_tables_d) - p->table_arena);
    memcpy(mirror, tables_host, total * 4);
    CU(cudaMemcpyAsync(pl->own_tables_d, mirror, total * 4, cudaMemcpyHostToDevice, s));
  } else {
    CU(cudaMemcpyAsync(pl->own_tables_d, tables_host, total * 4, cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));  // (arena exhausted: private allocation, no mirror — the caller's buffer must be read before we return)
  }
  p->n_memcpys++;
  pl->own_tables_set = true;
  return note_use(p, pl, s);
}

int kvpool_wait_offloads(kvpool_t* p, kvpool_placement_t* pl, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "wait_offloads: bad arguments");
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  for (auto& L : pl->layers) {
    if (L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
    if (L.ssd_stored) {  // the store commands of SSD-type devices complete on their workers: wait for the flags they raise
      const int rc = ssd_wait_stored(p, L, s);
      if (rc != KVPOOL_OK) return rc;
    }
  }
  return KVPOOL_OK;
}

int kvpool_synchronize(kvpool_t* p) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "synchronize: null pool");
  DeviceGuard guard(p->cuda_device);
  int rc = sync_pool_streams(p);
  if (rc == KVPOOL_OK && p->ssd_mask) rc = ssd_drain(p);  // and the workers of the SSD-type devices; EIO if a command failed
  if (rc != KVPOOL_OK) return rc;
  // offloads that have landed by now need no stream waits any more: later calls on those layers enqueue nothing but
  // their own work (which is what makes a zero-copy retrieve capturable into a CUDA graph)
  for (auto* pl : p->live)
    for (auto& L : pl->layers) settle_landed(L);
  return KVPOOL_OK;
}

int kvpool_pack(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, const void* k_base, const void* v_base, uint64_t stride,
                const int32_t* table, void* stage_dev, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
  if (L.map->K == 0) return KVPOOL_OK;
  if (!stage_dev || (reinterpret_cast<uintptr_t>(stage_dev) & 15u)) return fail(KVPOOL_EINVAL, "pack: stage_dev must be a 16-byte aligned device pointer");
  DeviceGuard guard(p->cuda_device);
  LayerArgs a = base_args(p, L, k_base, v_base, stride, table_of(pl, layer, table));
  for (uint32_t i = 0; i < p->n; ++i) a.pool_base[i] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(stage_dev) + static_cast<uint64_t>(L.map->start[i]) * p->payload);
  rc = launch_counted(p, a, true, false, static_cast<cudaStream_t>(cuda_stream));
  return rc == KVPOOL_OK ? note_use(p, pl, static_cast<cudaStream_t>(cuda_stream)) : rc;
}

int kvpool_unpack(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, void* k_base, void* v_base, uint64_t stride,
                  const int32_t* table, const void* stage_dev, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
  if (L.map->K == 0) return KVPOOL_OK;
  if (!stage_dev || (reinterpret_cast<uintptr_t>(stage_dev) & 15u)) return fail(KVPOOL_EINVAL, "unpack: stage_dev must be a 16-byte aligned device pointer");
  DeviceGuard guard(p->cuda_device);
  LayerArgs a = base_args(p, L, k_base, v_base, stride, table_of(pl, layer, table));
  for (uint32_t i = 0; i < p->n; ++i)
    a.pool_base[i] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(const_cast<void*>(stage_dev)) + static_cast<uint64_t>(L.map->start[i]) * p->payload);
  rc = launch_counted(p, a, false, false, static_cast<cudaStream_t>(cuda_stream));
  return rc == KVPOOL_OK ? note_use(p, pl, static_cast<cudaStream_t>(cuda_stream)) : rc;
}

}  // extern "C"
