// libkvpool.so, part 3 of 3: the development entry points of include/kvpool_dev.h — comparison baselines, consumer stand-ins,
// work counters and per-kernel profiling — and the counted / profiled launch wrappers the hot path goes through.
#include "kvpool_internal.hpp"

using namespace kvp;

namespace kvp {
namespace {

constexpr uint32_t kSpanCap = 16384;  // profiled launches between two reads that also get a device-clock span

// Hand the next launch its span pair (null once the arena is used up: such launches are timed by events only).
unsigned long long* take_span(kvpool* p, ProfRec* r) {
  if (!p->span_arena || p->span_cursor >= kSpanCap) return nullptr;
  r->span = static_cast<int32_t>(p->span_cursor++);
  return p->span_arena + 2ull * r->span;
}

// Spans start out as {UINT64_MAX, 0} so that atomicMin / atomicMax fold into them.
cudaError_t reset_spans(kvpool* p) {
  std::vector<unsigned long long> init(2ull * kSpanCap);
  for (uint32_t i = 0; i < kSpanCap; ++i) { init[2 * i] = ~0ull; init[2 * i + 1] = 0; }
  p->span_cursor = 0;
  cudaError_t e = cudaMemcpyAsync(p->span_arena, init.data(), init.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, p->upload);
  return e == cudaSuccess ? cudaStreamSynchronize(p->upload) : e;
}

cudaError_t prof_event(kvpool* p, cudaEvent_t* e) {
  if (!p->prof_free.empty()) { *e = p->prof_free.back(); p->prof_free.pop_back(); return cudaSuccess; }
  return cudaEventCreate(e);
}

// Profiled launches.  A TIMING event recorded on the launching stream holds that stream up until its timestamp has been
// written — 3 us on an idle GPU, 25 us under a concurrent host->GPU DMA, 47 us under a GPU->host one (measured on this
// box) — so an in-stream pair both delays the kernel and counts the delay.  Instead the stream gets two NON-timing
// markers (1 us each, unaffected by DMA) and the timing events are recorded on two side streams behind them: e0 on
// prof_s0 once the marker in front of the kernel has fired, e1 on prof_s1 once the marker behind it has.  The pair then
// spans the kernel (plus a few us of marker latency) and the launching stream is not held up at all.
int prof_side_streams(kvpool* p, cudaStream_t s, cudaStream_t* s0, cudaStream_t* s1) {
  auto it = p->prof_side.find(s);
  if (it == p->prof_side.end()) {
    std::pair<cudaStream_t, cudaStream_t> pr{nullptr, nullptr};
    CU(cudaStreamCreateWithFlags(&pr.first, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&pr.second, cudaStreamNonBlocking));
    it = p->prof_side.emplace(s, pr).first;
  }
  *s0 = it->second.first;
  *s1 = it->second.second;
  return KVPOOL_OK;
}
int prof_begin(kvpool* p, ProfRec* r, cudaStream_t s) {
  CU(prof_event(p, &r->e0));
  CU(prof_event(p, &r->e1));
  if (p->prof_instream) { CU(cudaEventRecord(r->e0, s)); return KVPOOL_OK; }
  cudaStream_t s0 = nullptr, s1 = nullptr;
  const int rc = prof_side_streams(p, s, &s0, &s1);
  if (rc != KVPOOL_OK) return rc;
  cudaEvent_t m = nullptr;
  CU(take_event(p, &m));
  CU(cudaEventRecord(m, s));
  CU(cudaStreamWaitEvent(s0, m, 0));
  p->ev_free.push_back(m);  // the wait has captured this record; a later re-record does not move it
  CU(cudaEventRecord(r->e0, s0));
  return KVPOOL_OK;
}
int prof_end(kvpool* p, ProfRec* r, cudaStream_t s) {
  if (p->prof_instream) { CU(cudaEventRecord(r->e1, s)); }
  else {
    cudaStream_t s0 = nullptr, s1 = nullptr;
    const int rc = prof_side_streams(p, s, &s0, &s1);
    if (rc != KVPOOL_OK) return rc;
    cudaEvent_t m = nullptr;
    CU(take_event(p, &m));
    CU(cudaEventRecord(m, s));
    CU(cudaStreamWaitEvent(s1, m, 0));
    p->ev_free.push_back(m);
    CU(cudaEventRecord(r->e1, s1));
  }
  p->prof.push_back(*r);
  return KVPOOL_OK;
}

}  // namespace

// Launch one layer kernel, counted and (when profiling) bracketed by an event pair.
int launch_counted(kvpool* p, const LayerArgs& a, bool pack, bool link_bound, cudaStream_t s, bool lane) {
  ProfRec r;
  if (p->profiling) {
    r.bytes = static_cast<uint64_t>(a.K) * p->payload;
    r.kind = (link_bound ? 2 : 0) + (pack ? 0 : 1);
    const int rc = prof_begin(p, &r, s);
    if (rc != KVPOOL_OK) return rc;
  }
  LayerArgs timed = a;
  if (p->profiling) timed.span = take_span(p, &r);
  CU(launch_layer_copy(timed, pack, launch_cfg(p, link_bound, pack, lane), s));
  p->n_kernels++;
  if (p->profiling) return prof_end(p, &r, s);
  return KVPOOL_OK;
}

// One multi-layer launch, counted and (when profiling) bracketed by an event pair on `s`.
int launch_multi_counted(kvpool* p, const MultiArgs& ma, bool pack, bool link_bound, cudaStream_t s) {
  ProfRec r;
  if (p->profiling) {
    r.bytes = static_cast<uint64_t>(ma.total_units) * p->payload;
    r.kind = (link_bound ? 2 : 0) + (pack ? 0 : 1);
    const int rc = prof_begin(p, &r, s);
    if (rc != KVPOOL_OK) return rc;
  }
  MultiArgs timed = ma;
  if (p->profiling) timed.span = take_span(p, &r);
  LaunchCfg cfg = launch_cfg(p, link_bound, pack);
  // a signalled retrieve runs the 16-byte kernel (kernels.cu): 8 CTAs of it fill the link (profiles/r1_sweep_link.txt)
  if (ma.sig_flag && link_bound && !p->hbm_mask) cfg.ctas = std::max<uint32_t>(cfg.ctas, 8);
  CU(launch_multi_copy(timed, pack, cfg, s));
  p->n_kernels++;
  if (p->profiling) return prof_end(p, &r, s);
  return KVPOOL_OK;
}

}  // namespace kvp

extern "C" {

// Baseline for comparison: 2*K_l individual cudaMemcpyAsync calls per layer, no kernel.
static int naive_layer(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, bool pack, const void* k_base, const void* v_base, uint64_t stride,
                       const int32_t* table_host, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table_host);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
  if (p->ssd_mask) return fail(KVPOOL_EINVAL, "the per-block memcpy baseline has no SSD branch");
  if (!pack && !L.offloaded) return fail(KVPOOL_ESTATE, "retrieve: layer %u was never offloaded", layer);
  if (pack) { L.offloaded = true; L.have.clear(); }
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
  for (uint64_t j = 0; j < L.map->K; ++j) {
    const uint32_t d = L.map->dev[j];
    uint8_t* pooled = pool_bytes(p, d) + L.stripe_off[d] + static_cast<uint64_t>(L.map->slot[j]) * p->payload;
    uint8_t* kb = static_cast<uint8_t*>(const_cast<void*>(k_base)) + static_cast<uint64_t>(table_host[j]) * stride;
    uint8_t* vb = static_cast<uint8_t*>(const_cast<void*>(v_base)) + static_cast<uint64_t>(table_host[j]) * stride;
    if (pack) {
      CU(cudaMemcpyAsync(pooled, kb, p->kvb, cudaMemcpyDefault, s));
      CU(cudaMemcpyAsync(pooled + p->kvb, vb, p->kvb, cudaMemcpyDefault, s));
    } else {
      CU(cudaMemcpyAsync(kb, pooled, p->kvb, cudaMemcpyDefault, s));
      CU(cudaMemcpyAsync(vb, pooled + p->kvb, p->kvb, cudaMemcpyDefault, s));
    }
    p->n_memcpys += 2;
  }
  if (pack && L.map->K) {
    CU(cudaEventRecord(L.landed, s));
    L.landed_pending = true;
  }
  return note_use(p, pl, s);
}

int kvpool_offload_naive(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, const void* k_base, const void* v_base, uint64_t stride,
                         const int32_t* table_host, void* cuda_stream) {
  return naive_layer(p, pl, layer, true, k_base, v_base, stride, table_host, cuda_stream);
}

int kvpool_retrieve_naive(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, void* k_base, void* v_base, uint64_t stride,
                          const int32_t* table_host, void* cuda_stream) {
  return naive_layer(p, pl, layer, false, k_base, v_base, stride, table_host, cuda_stream);
}

int kvpool_checksum(kvpool_t* p, const void* k_base, const void* v_base, uint64_t stride, const int32_t* table, uint32_t n_blocks,
                    uint64_t* sum_dev, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !sum_dev) return fail(KVPOOL_EINVAL, "checksum: null argument");
  if (n_blocks == 0) return KVPOOL_OK;
  if (!k_base || !v_base || !table) return fail(KVPOOL_EINVAL, "checksum: null k_base / v_base / block table");
  if ((reinterpret_cast<uintptr_t>(k_base) | reinterpret_cast<uintptr_t>(v_base) | stride) & 15u)
    return fail(KVPOOL_EINVAL, "checksum: k_base, v_base and block_stride_bytes must be multiples of 16");
  if (reinterpret_cast<uintptr_t>(sum_dev) & 7u) return fail(KVPOOL_EINVAL, "checksum: sum_dev must be 8-byte aligned");
  DeviceGuard guard(p->cuda_device);
  CU(launch_checksum(static_cast<const uint8_t*>(k_base), static_cast<const uint8_t*>(v_base), stride, table, n_blocks,
                     static_cast<uint32_t>(p->kvb), reinterpret_cast<unsigned long long*>(sum_dev), p->tune.hbm_ctas,
                     static_cast<cudaStream_t>(cuda_stream)));
  p->n_kernels++;
  return KVPOOL_OK;
}

int kvpool_checksum_layers(kvpool_t* p, uint32_t n_layers, const void* const* k_bases, const void* const* v_bases, uint64_t stride,
                           const int32_t* const* tables, const uint32_t* n_blocks, void* const* layer_ready, uint64_t* sums_dev,
                           void* cuda_stream) {
  PoolLock lock__(p);
  if (!p || !k_bases || !v_bases || !tables || !n_blocks || !sums_dev) return fail(KVPOOL_EINVAL, "checksum_layers: null argument");
  DeviceGuard guard(p->cuda_device);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  for (uint32_t q = 0; q < n_layers; ++q) {
    if (layer_ready && layer_ready[q]) CU(cudaStreamWaitEvent(s, static_cast<cudaEvent_t>(layer_ready[q]), 0));
    const int rc = kvpool_checksum(p, k_bases[q], v_bases[q], stride, tables[q], n_blocks[q], sums_dev + q, s);
    if (rc != KVPOOL_OK) return rc;
  }
  return KVPOOL_OK;
}

int kvpool_spin(kvpool_t* p, uint64_t ns, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "spin: null pool");
  if (ns > 10ull * 1000 * 1000 * 1000) return fail(KVPOOL_EINVAL, "spin: more than 10 s");
  DeviceGuard guard(p->cuda_device);
  CU(launch_spin(ns, static_cast<cudaStream_t>(cuda_stream)));
  p->n_kernels++;
  return KVPOOL_OK;
}

int kvpool_set_profiling(kvpool_t* p, int enabled) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "set_profiling: null pool");
  if (enabled < 0 || enabled > KVPOOL_PROFILE_INSTREAM) return fail(KVPOOL_EINVAL, "set_profiling: mode %d", enabled);
  if (enabled && !p->span_arena) {
    DeviceGuard guard(p->cuda_device);
    CU(cudaMalloc(reinterpret_cast<void**>(&p->span_arena), 2ull * kSpanCap * sizeof(unsigned long long)));
    CU(reset_spans(p));
  }
  p->profiling = enabled != 0;
  p->prof_instream = enabled == KVPOOL_PROFILE_INSTREAM;
  return KVPOOL_OK;
}

int kvpool_profile_read_clock(kvpool_t* p, int kind, double* total_ms, double* device_ms, uint64_t* launches, uint64_t* device_launches,
                              uint64_t* bytes) {
  PoolLock lock__(p);
  if (!p || kind < 0 || kind > 3) return fail(KVPOOL_EINVAL, "profile_read: bad arguments");
  DeviceGuard guard(p->cuda_device);
  double ms_sum = 0, dev_ms_sum = 0;
  uint64_t n = 0, n_dev = 0, b = 0;
  std::vector<ProfRec> keep;
  std::vector<unsigned long long> spans;
  bool any_span = false;
  for (auto& r : p->prof)
    if (r.kind == kind) {
      CU(cudaEventSynchronize(r.e0));
      CU(cudaEventSynchronize(r.e1));
      any_span |= r.span >= 0;
    }
  if (any_span) {  // every launch of this kind has completed: one read-back of the spans handed out so far
    spans.resize(2ull * p->span_cursor);
    CU(cudaMemcpyAsync(spans.data(), p->span_arena, spans.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->upload));
    CU(cudaStreamSynchronize(p->upload));
  }
  for (auto& r : p->prof) {
    if (r.kind != kind) { keep.push_back(r); continue; }
    float ms = 0;
    CU(cudaEventElapsedTime(&ms, r.e0, r.e1));
    ms_sum += ms;
    n += 1;
    b += r.bytes;
    if (r.span >= 0) {
      const unsigned long long t0 = spans[2ull * r.span], t1 = spans[2ull * r.span + 1];
      if (t1 >= t0) { dev_ms_sum += static_cast<double>(t1 - t0) * 1e-6; n_dev += 1; }  // (a launch with no work leaves {max, 0})
    }
    p->prof_free.push_back(r.e0);
    p->prof_free.push_back(r.e1);
  }
  p->prof.swap(keep);
  if (p->prof.empty() && p->span_arena && p->span_cursor) CU(reset_spans(p));  // all read: the arena starts over
  if (total_ms) *total_ms = ms_sum;
  if (device_ms) *device_ms = dev_ms_sum;
  if (launches) *launches = n;
  if (device_launches) *device_launches = n_dev;
  if (bytes) *bytes = b;
  return KVPOOL_OK;
}

int kvpool_profile_read(kvpool_t* p, int kind, double* total_ms, uint64_t* launches, uint64_t* bytes) {
  return kvpool_profile_read_clock(p, kind, total_ms, nullptr, launches, nullptr, bytes);
}

int kvpool_stats(const kvpool_t* p, uint64_t* kernel_launches, uint64_t* memcpy_calls) {
  if (!p) return fail(KVPOOL_EINVAL, "stats: null pool");
  if (kernel_launches) *kernel_launches = p->n_kernels;
  if (memcpy_calls) *memcpy_calls = p->n_memcpys;
  return KVPOOL_OK;
}

}  // extern "C"
