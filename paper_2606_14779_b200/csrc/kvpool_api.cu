// C ABI of libkvpool (include/kvpool.h; development entry points: include/kvpool_dev.h): pool life cycle, placement + GLT, and the per-layer
// offload / retrieve choreography over CUDA streams and events.  Device code lives in kernels.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <memory>
#include <mutex>
#include <numeric>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/kvpool.h"
#include "../../include/kvpool_dev.h"
#include "kernels.cuh"
#include "placement.hpp"
#include "pool_mem.hpp"

using namespace kvp;

static_assert(KVPOOL_MAX_DEVICES == kvp::kMaxDevices && KVPOOL_MAX_DEVICES == kvp::kMaxDev, "device limit mismatch");

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

#define CU(call)                                                                              \
  do {                                                                                        \
    cudaError_t e__ = (call);                                                                 \
    if (e__ != cudaSuccess) return fail(KVPOOL_ECUDA, "%s: %s", #call, cudaGetErrorString(e__)); \
  } while (0)

struct DeviceGuard {  // make the pool's GPU current for the duration of a call
  int prev = -1;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// Serialises host threads on one pool (null-tolerant so that it can precede the argument checks; recursive because the
// batched calls go through the per-layer entry points).
struct PoolLock {
  std::unique_lock<std::recursive_mutex> l;
  explicit PoolLock(kvpool* p);
};

// Dense per-layer GLT columns shared by all layers of a placement that move the same number of blocks.
struct LayerMap {
  uint64_t K = 0;
  std::vector<uint32_t> counts;   // [N]
  std::vector<uint32_t> start;    // [N] first stripe-order position of device i (prefix sum of counts)
  std::vector<uint8_t> dev;       // [K]
  std::vector<uint32_t> slot;     // [K]
  std::vector<uint32_t> order;    // [K] order[start[i] + s] = logical block stored at slot s of device i (ascending in s)
  const uint8_t* dev_d = nullptr; // device copies
  const uint32_t* slot_d = nullptr;
  const uint32_t* order_d = nullptr;
  const uint32_t* visit_d = nullptr; // mixed pools only: the layer's blocks with those of host-memory devices first (kernels.cuh)
  uint64_t host_blocks = 0;       // blocks of the layer that sit on host-memory devices (the rest: HBM-type devices)
};

struct LayerState {
  std::shared_ptr<LayerMap> map;
  std::vector<uint64_t> stripe_off;  // [N] byte offset of this layer's stripe inside pool buffer i
  const uint64_t* base_d = nullptr;  // device: [N] GPU-visible addresses of this layer's stripes (for batched launches)
  bool offloaded = false;            // every block of the layer has been offloaded at least once
  std::vector<uint64_t> have;        // else, once a partial offload has happened: bit j = logical block j is in the pool
  cudaEvent_t landed = nullptr;      // recorded when the layer's stripes are complete in the pool
  bool landed_pending = false;
};

struct ProfRec {  // one profiled kernel launch
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  uint64_t bytes = 0;
  int kind = 0;
  int32_t span = -1;  // index of the launch's {min start, max end} pair in the pool's span arena, -1 = none left
};

struct StageSlot {
  uint8_t* buf = nullptr;
  cudaEvent_t kernel_done = nullptr;          // last kernel that read/wrote the slot
  cudaEvent_t gate = nullptr;                 // scratch: fans one stream's waits out to the other I/O streams
  uint32_t copies_after_kernel = 0;           // devices whose copy_done must also be awaited before reuse: set by an
                                              // offload (D2H copies follow the pack); a retrieve's copies precede its
                                              // unpack, so kernel_done alone covers them
  std::vector<cudaEvent_t> copy_done;         // [N] last memcpy per pool stream that read/wrote the slot
};

}  // namespace

struct GltHash {  // Table I `key`: splitmix64 finaliser of the identifier
  static uint64_t mix(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  }
  size_t operator()(uint64_t id) const { return static_cast<size_t>(mix(id)); }
};
struct GltRef {
  kvpool_placement* pl;
  uint32_t layer, block;
};

struct kvpool_placement {
  kvpool* pool = nullptr;
  std::vector<uint64_t> bound_ids;  // identifiers bound through kvpool_glt_bind, erased at release
  std::vector<LayerState> layers;
  std::vector<uint64_t> region_off, region_bytes;  // [N] one contiguous region per pool device holds all layers' stripes
  uint8_t* tables_d = nullptr;   // every LayerMap's dev/slot columns, contiguous
  uint64_t tables_bytes = 0;
  bool tables_in_arena = false;  // carved out of the pool's table arena (else a private cudaMalloc)
  // last work enqueued with this placement on each caller stream (non-timing events): kvpool_release waits for them, so
  // that stripes never go back to the allocator while a kernel on a caller's stream still reads or writes them
  std::vector<std::pair<cudaStream_t, cudaEvent_t>> last_use;
  // kvpool_set_tables: the request's block tables, uploaded in one copy; layer l's table starts at own_table_off[l] entries
  int32_t* own_tables_d = nullptr;
  uint64_t own_tables_bytes = 0;
  bool own_tables_in_arena = false, own_tables_set = false;
  std::vector<uint64_t> own_table_off;
};

struct kvpool {
  int cuda_device = 0;
  int sm_count = 148;
  kvpool_geometry geom{};
  uint64_t kvb = 0, payload = 0;
  uint32_t n = 0;
  std::vector<double> bandwidth;
  std::vector<uint64_t> w;
  std::vector<HostBuffer> bufs;
  std::vector<uint32_t> link_group;  // [N] kvpool_device_desc.link_group: devices of one group share io / io_out streams
  std::vector<cudaStream_t> own_streams;  // every stream created for io / io_out, once (members of a group alias one)
  uint32_t hbm_mask = 0;  // bit i: pool device i is GPU memory (KVPOOL_DEV_HBM): reached by the kernels directly, never staged or copied
  std::vector<StripeAllocator> alloc;
  std::vector<cudaStream_t> io;      // one I/O stream per pool device ("independent I/O streams"): host -> GPU copies
  cudaStream_t join_out = nullptr;   // gathers an offload's copies for its `landed` event; carries no work of its own
  std::vector<cudaStream_t> io_out;  // and one for GPU -> host copies, so that an offload and a retrieve use both directions of the link at once
  std::vector<StageSlot> slots;
  uint64_t slot_bytes = 0;
  uint64_t slot_cursor = 0;
  uint8_t* table_arena = nullptr;  // device memory for placements' GLT columns: no cudaMalloc/cudaFree per request
  uint8_t* table_arena_host = nullptr;  // its pinned host mirror: tables are built in place and uploaded on `upload`
  cudaStream_t upload = nullptr;   // the library's own non-blocking stream for table uploads and small read-backs, so that
                                   // kvpool_place never touches the legacy default stream (which would make it wait for
                                   // whatever the application has queued there)
  StripeAllocator table_alloc;
  std::vector<cudaEvent_t> ev_free;  // recycled cudaEventDisableTiming events
  int path = KVPOOL_PATH_AUTO;
  kvpool_tuning tune{};
  std::vector<kvpool_placement*> live;
  std::unordered_map<uint64_t, GltRef, GltHash> glt;  // keyed GLT: identifier -> (placement, layer, block)
  uint32_t check_nphys = 0;              // kvpool_set_table_check: the kernels skip and count table entries outside [0, check_nphys)
  unsigned long long* bad_d = nullptr;   // device counter of such entries
  uint64_t n_kernels = 0, n_memcpys = 0;
  bool profiling = false;
  bool prof_instream = false;            // KVPOOL_PROFILE_INSTREAM: timing events on the launching stream itself (perturbs it, see prof_begin)
  // side streams that carry the timing events of profiled launches: one pair per launching stream, so that the e0 of one
  // caller stream never queues behind another caller stream's marker wait
  std::unordered_map<cudaStream_t, std::pair<cudaStream_t, cudaStream_t>> prof_side;
  std::vector<ProfRec> prof;
  std::vector<cudaEvent_t> prof_free;  // timing events ready for reuse
  unsigned long long* span_arena = nullptr;  // device: kSpanCap x {min start, max end} in %globaltimer ns, written by the kernels
  uint32_t span_cursor = 0;
  std::recursive_mutex mu;  // every entry point that touches pool state holds it: calls only enqueue work, so the lock is short
};

namespace {

PoolLock::PoolLock(kvpool* p) {
  if (p) l = std::unique_lock<std::recursive_mutex>(p->mu);
}

void default_tuning(kvpool* p) {
  p->tune.kernel = KVPOOL_KERNEL_VEC16;
  p->tune.link_kernel = KVPOOL_KERNEL_BULK;  // 2 CTAs already saturate the link (profiles/r1_sweep_link.txt)
  p->tune.hbm_ctas = 16u * p->sm_count;  // many short CTAs balance the tail better than a persistent grid here (profiles/r1_sweep_hbm.txt)
  p->tune.link_ctas = 4;
  p->tune.bulk_chunk = 16384;
  p->tune.bulk_stages = 6;
  p->tune.bulk_warps = 2;
  p->tune.stage_slots = 2;                   // one slot fills while the other drains; the kernels take ~2 % of a copy's time
  p->tune.stage_chunk_bytes = 256ull << 20;  // ring <= 512 MiB whatever the context length (larger layers: device-major chunks)
  p->tune.vec_threads = 512;
  p->tune.vec_unroll = 8;
  p->tune.group_bytes = 64ull << 20;
  p->tune.auto_threshold_bytes = 8ull << 20;
  p->tune.pdl = 1;
}

void free_slots(kvpool* p) {
  for (auto& s : p->slots) {
    if (s.buf) cudaFree(s.buf);
    if (s.kernel_done) cudaEventDestroy(s.kernel_done);
    if (s.gate) cudaEventDestroy(s.gate);
    for (auto e : s.copy_done) cudaEventDestroy(e);
  }
  p->slots.clear();
  p->slot_bytes = 0;
}

int sync_pool_streams(kvpool* p) {
  for (auto s : p->own_streams) CU(cudaStreamSynchronize(s));
  if (p->join_out) CU(cudaStreamSynchronize(p->join_out));
  return KVPOOL_OK;
}

// (Re)build the staging ring so that every slot holds `bytes`.  Not on the hot path (called from place).
int ensure_slots(kvpool* p, uint64_t bytes) {
  if (bytes <= p->slot_bytes && p->slots.size() == p->tune.stage_slots) return KVPOOL_OK;
  CU(cudaDeviceSynchronize());
  const uint64_t want = std::max(bytes, p->slot_bytes);
  free_slots(p);
  p->slots.resize(p->tune.stage_slots);
  for (auto& s : p->slots) {
    if (want > 0) {
      cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&s.buf), want);
      if (e != cudaSuccess) {
        cudaGetLastError();
        free_slots(p);
        return fail(KVPOOL_ENOMEM, "staging slot of %llu bytes: %s", (unsigned long long)want, cudaGetErrorString(e));
      }
    }
    CU(cudaEventCreateWithFlags(&s.kernel_done, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&s.gate, cudaEventDisableTiming));
    s.copy_done.resize(p->n);
    for (auto& e : s.copy_done) CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  p->slot_bytes = want;
  return KVPOOL_OK;
}

bool is_live(const kvpool* p, const kvpool_placement* pl) {
  return std::find(p->live.begin(), p->live.end(), pl) != p->live.end();
}

constexpr uint64_t kTableArenaBytes = 8ull << 20;

void free_tables(kvpool* p, kvpool_placement* pl) {
  if (pl->own_tables_d) {
    if (pl->own_tables_in_arena) p->table_alloc.free(static_cast<uint64_t>(reinterpret_cast<uint8_t*>(pl->own_tables_d) - p->table_arena), pl->own_tables_bytes);
    else cudaFree(pl->own_tables_d);
    pl->own_tables_d = nullptr;
    pl->own_tables_set = false;
  }
  if (!pl->tables_d) return;
  if (pl->tables_in_arena) p->table_alloc.free(static_cast<uint64_t>(pl->tables_d - p->table_arena), pl->tables_bytes);
  else cudaFree(pl->tables_d);
  pl->tables_d = nullptr;
}

cudaError_t take_event(kvpool* p, cudaEvent_t* e) {
  if (!p->ev_free.empty()) { *e = p->ev_free.back(); p->ev_free.pop_back(); return cudaSuccess; }
  return cudaEventCreateWithFlags(e, cudaEventDisableTiming);
}

// Remember that `s` carries work of this placement (skipped while `s` is being captured into a CUDA graph: a captured
// event could not be waited for later, and a graph's lifetime is the caller's business, kvpool.h).
int note_use(kvpool* p, kvpool_placement* pl, cudaStream_t s) {
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(s, &st) != cudaSuccess) { cudaGetLastError(); return KVPOOL_OK; }
  if (st != cudaStreamCaptureStatusNone) return KVPOOL_OK;
  for (auto& u : pl->last_use)
    if (u.first == s) { CU(cudaEventRecord(u.second, s)); return KVPOOL_OK; }
  cudaEvent_t e = nullptr;
  CU(take_event(p, &e));
  pl->last_use.emplace_back(s, e);
  CU(cudaEventRecord(e, s));
  return KVPOOL_OK;
}

void destroy_placement(kvpool* p, kvpool_placement* pl) {
  for (uint64_t id : pl->bound_ids) p->glt.erase(id);
  for (auto& u : pl->last_use) p->ev_free.push_back(u.second);
  for (uint32_t i = 0; i < p->n && i < pl->region_off.size(); ++i) p->alloc[i].free(pl->region_off[i], pl->region_bytes[i]);
  for (auto& L : pl->layers)
    if (L.landed) p->ev_free.push_back(L.landed);
  free_tables(p, pl);
  delete pl;
}

int check_layer_call(kvpool* p, kvpool_placement* pl, uint32_t layer, const void* k_base, const void* v_base, uint64_t stride,
                     const int32_t* table) {
  if (!p || !pl) return fail(KVPOOL_EINVAL, "null pool or placement");
  if (pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "placement does not belong to this pool");
  if (layer >= p->geom.n_layers) return fail(KVPOOL_EINVAL, "layer %u out of range (n_layers %u)", layer, p->geom.n_layers);
  if (pl->layers[layer].map->K == 0) return KVPOOL_OK;
  if (!k_base || !v_base) return fail(KVPOOL_EINVAL, "null k_base / v_base");
  if (!table && !pl->own_tables_set) return fail(KVPOOL_EINVAL, "null block table (and no tables uploaded with kvpool_set_tables)");
  if ((reinterpret_cast<uintptr_t>(k_base) | reinterpret_cast<uintptr_t>(v_base) | stride) & 15u)
    return fail(KVPOOL_EINVAL, "k_base, v_base and block_stride_bytes must be multiples of 16");
  if (stride < p->kvb) return fail(KVPOOL_EINVAL, "block_stride_bytes %llu < block bytes %llu", (unsigned long long)stride,
                                   (unsigned long long)p->kvb);
  return KVPOOL_OK;
}

// The layer's block table on the device: the caller's, or (null) the one kvpool_set_tables uploaded.
inline const int32_t* table_of(const kvpool_placement* pl, uint32_t layer, const int32_t* given) {
  return given ? given : pl->own_tables_d + pl->own_table_off[layer];
}

LayerArgs base_args(const kvpool* p, const LayerState& L, const void* k_base, const void* v_base, uint64_t stride,
                    const int32_t* table) {
  LayerArgs a{};
  a.k_base = static_cast<uint8_t*>(const_cast<void*>(k_base));
  a.v_base = static_cast<uint8_t*>(const_cast<void*>(v_base));
  a.stride = stride;
  a.table = table;
  a.dev = L.map->dev_d;
  a.slot = L.map->slot_d;
  a.K = static_cast<uint32_t>(L.map->K);
  a.j0 = 0;
  a.kvb = static_cast<uint32_t>(p->kvb);
  a.nphys_check = p->check_nphys;
  a.bad = p->bad_d;
  return a;
}

inline bool is_hbm(const kvpool* p, uint32_t i) { return (p->hbm_mask >> i) & 1u; }
// Where the CPU / copy engines find pool device i's bytes: the host address, or the device pointer of an HBM device.
inline uint8_t* pool_bytes(const kvpool* p, uint32_t i) {
  return static_cast<uint8_t*>(is_hbm(p, i) ? p->bufs[i].dev_alias : p->bufs[i].host);
}

LaunchCfg launch_cfg(const kvpool* p, bool link_bound, bool pack = false) {
  // a zero-copy launch over a pool with HBM devices moves most of its bytes at HBM / NVLink rates: give it the HBM grid
  if (p->hbm_mask) link_bound = false;
  LaunchCfg c{};
  c.kernel = link_bound ? p->tune.link_kernel : p->tune.kernel;
  c.ctas = link_bound ? p->tune.link_ctas : p->tune.hbm_ctas;
  // the hybrid path is made for both directions of the link at once: under a concurrent host->GPU copy stream the posted
  // writes of 4 CTAs reach 43.8 GB/s, those of 8 CTAs 45.8 (profiles/r2_duplex.md)
  if (link_bound && pack && p->path == KVPOOL_PATH_HYBRID) c.ctas = std::max<uint32_t>(c.ctas, 8);
  c.bulk_chunk = p->tune.bulk_chunk;
  c.bulk_stages = p->tune.bulk_stages;
  c.bulk_warps = p->tune.bulk_warps;
  c.vec_threads = p->tune.vec_threads;
  c.vec_unroll = p->tune.vec_unroll;
  c.sm_count = static_cast<uint32_t>(p->sm_count);
  c.pdl = p->tune.pdl != 2;
  return c;
}

inline bool all_hbm(const kvpool* p) { return p->hbm_mask == (p->n >= 32 ? 0xFFFFFFFFu : (1u << p->n) - 1u); }

// Does a transfer of `host_bytes` to / from host-memory devices go through the staging ring and the copy engines?
bool use_staged(const kvpool* p, bool pack, uint64_t host_bytes) {
  if (all_hbm(p)) return false;   // nothing to stage: every stripe is reached in place (one kernel, HBM grid)
  if (host_bytes == 0) return false;  // all of its blocks went to HBM-type devices (tiny K, large weights)
  switch (p->path) {
    case KVPOOL_PATH_ZEROCOPY: return false;
    case KVPOOL_PATH_STAGED: return true;
    case KVPOOL_PATH_HYBRID:
      if (pack) return false;  // offload by the kernel's own stores, retrieve as on the auto path
      [[fallthrough]];
    default:
      // judged by what would travel through the copy engines: in a pool with HBM-type devices the host devices' share of a
      // layer is small (Eq. 1 gives a 55 GB/s link 2 % next to 3 TB/s of HBM); below the threshold the same kernel that
      // reaches the HBM stripes in place also stores / loads the mapped host stripes, instead of a few latency-bound copies
      return host_bytes >= p->tune.auto_threshold_bytes;
  }
}

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

// Launch one layer kernel, counted and (when profiling) bracketed by an event pair.
int launch_counted(kvpool* p, const LayerArgs& a, bool pack, bool link_bound, cudaStream_t s) {
  ProfRec r;
  if (p->profiling) {
    r.bytes = static_cast<uint64_t>(a.K) * p->payload;
    r.kind = (link_bound ? 2 : 0) + (pack ? 0 : 1);
    const int rc = prof_begin(p, &r, s);
    if (rc != KVPOOL_OK) return rc;
  }
  LayerArgs timed = a;
  if (p->profiling) timed.span = take_span(p, &r);
  CU(launch_layer_copy(timed, pack, launch_cfg(p, link_bound, pack), s));
  p->n_kernels++;
  if (p->profiling) return prof_end(p, &r, s);
  return KVPOOL_OK;
}

// Make `s` wait until the previous user of a staging slot is done with it.
int wait_slot_free(kvpool* p, StageSlot& slot, cudaStream_t s) {
  CU(cudaStreamWaitEvent(s, slot.kernel_done, 0));
  for (uint32_t i = 0; i < p->n; ++i)
    if (slot.copies_after_kernel >> i & 1u) CU(cudaStreamWaitEvent(s, slot.copy_done[i], 0));
  return KVPOOL_OK;
}

// An offload that has certainly landed needs no further stream waits.
void settle_landed(LayerState& L) {
  if (!L.landed_pending) return;
  if (cudaEventQuery(L.landed) == cudaSuccess) L.landed_pending = false;
  else cudaGetLastError();  // cudaErrorNotReady is not an error
}

}  // namespace

extern "C" {

const char* kvpool_last_error(void) { return g_err.c_str(); }
const char* kvpool_version(void) { return "kvpool 0.1 (sm_100a)"; }

int kvpool_plan_weights(const double* b, uint32_t n, uint64_t* w_out) {
  if (!b || !w_out || n == 0 || n > KVPOOL_MAX_DEVICES) return fail(KVPOOL_EINVAL, "plan_weights: bad arguments");
  if (!quantise_weights(b, n, w_out)) return fail(KVPOOL_EINVAL, "bandwidth must be positive and at least 0.0005 GB/s");
  return KVPOOL_OK;
}

int kvpool_plan_layer(const uint64_t* w, uint32_t n, uint64_t K, uint32_t* counts_out, uint8_t* dev_out, uint32_t* slot_out) {
  if (!w || !counts_out || n == 0 || n > KVPOOL_MAX_DEVICES || K > 0xFFFFFFFFull) return fail(KVPOOL_EINVAL, "plan_layer: bad arguments");
  if ((dev_out == nullptr) != (slot_out == nullptr)) return fail(KVPOOL_EINVAL, "plan_layer: dev_out and slot_out go together");
  for (uint32_t i = 0; i < n; ++i)
    if (w[i] == 0) return fail(KVPOOL_EINVAL, "plan_layer: weight %u is zero", i);
  target_counts(w, n, K, counts_out);
  if (dev_out) wrr_closed_form(counts_out, n, K, dev_out, slot_out);
  return KVPOOL_OK;
}

int kvpool_validate_table(const int32_t* table, uint64_t K, uint64_t nphys) {
  if (K == 0) return KVPOOL_OK;
  if (!table) return fail(KVPOOL_EINVAL, "validate_table: null table");
  if (nphys == 0 || nphys > 0x7fffffffull) return fail(KVPOOL_EINVAL, "validate_table: nphys %llu not in 1..2^31-1", (unsigned long long)nphys);
  if (K > nphys) return fail(KVPOOL_EINVAL, "validate_table: %llu entries cannot be distinct among %llu physical blocks", (unsigned long long)K, (unsigned long long)nphys);
  std::vector<uint64_t> seen((nphys + 63) / 64, 0);
  for (uint64_t j = 0; j < K; ++j) {
    const int64_t v = table[j];
    if (v < 0 || static_cast<uint64_t>(v) >= nphys) return fail(KVPOOL_EINVAL, "validate_table: entry %llu = %lld is outside [0, %llu)", (unsigned long long)j, (long long)v, (unsigned long long)nphys);
    uint64_t& word = seen[static_cast<uint64_t>(v) >> 6];
    const uint64_t bit = 1ull << (v & 63);
    if (word & bit) return fail(KVPOOL_EINVAL, "validate_table: physical block %lld appears twice (second time at entry %llu)", (long long)v, (unsigned long long)j);
    word |= bit;
  }
  return KVPOOL_OK;
}

int kvpool_create(const kvpool_device_desc* devs, uint32_t n_devs, const kvpool_geometry* g, int cuda_device, uint32_t flags,
                  kvpool_t** out) {
  if (!devs || !g || !out) return fail(KVPOOL_EINVAL, "create: null argument");
  *out = nullptr;
  if (flags != 0) return fail(KVPOOL_EINVAL, "create: unknown flags 0x%x", flags);
  if (n_devs == 0 || n_devs > KVPOOL_MAX_DEVICES) return fail(KVPOOL_EINVAL, "create: n_devs %u not in 1..%u", n_devs, KVPOOL_MAX_DEVICES);
  if (!g->n_layers || !g->block_tokens || !g->n_kv_heads || !g->head_dim || !g->elem_bytes) return fail(KVPOOL_EINVAL, "create: zero in geometry");
  const uint64_t kvb = static_cast<uint64_t>(g->block_tokens) * g->n_kv_heads * g->head_dim * g->elem_bytes;
  if (kvb % 16 != 0 || kvb > (1ull << 30)) return fail(KVPOOL_EINVAL, "create: block bytes %llu must be a multiple of 16 and <= 1 GiB", (unsigned long long)kvb);
  std::vector<double> bw(n_devs);
  std::vector<uint64_t> w(n_devs);
  for (uint32_t i = 0; i < n_devs; ++i) {
    bw[i] = devs[i].bandwidth_gbps;
    if (devs[i].capacity_bytes == 0) return fail(KVPOOL_EINVAL, "create: device %u has zero capacity", i);
    if (devs[i].flags & ~(KVPOOL_DEV_WRITE_COMBINED | KVPOOL_DEV_NUMA_STRICT | KVPOOL_DEV_HBM | KVPOOL_DEV_CUDA_HOSTALLOC)) return fail(KVPOOL_EINVAL, "create: device %u unknown flags", i);
    if ((devs[i].flags & KVPOOL_DEV_HBM) && (devs[i].flags & ~KVPOOL_DEV_HBM)) return fail(KVPOOL_EINVAL, "create: device %u: KVPOOL_DEV_HBM excludes the host-memory flags", i);
    if (devs[i].numa_node < KVPOOL_NUMA_AUTO) return fail(KVPOOL_EINVAL, "create: device %u: numa_node %d", i, devs[i].numa_node);
  }
  if (!quantise_weights(bw.data(), n_devs, w.data())) return fail(KVPOOL_EINVAL, "create: bandwidth must be positive (>= 0.0005 GB/s)");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(KVPOOL_ECUDA, "create: no CUDA device (this library has no CPU fallback)");
  }
  if (cuda_device < 0 || cuda_device >= ndev) return fail(KVPOOL_EINVAL, "create: cuda_device %d out of range", cuda_device);
  DeviceGuard guard(cuda_device);
  CU(cudaFree(nullptr));
  CU(kernels_init());

  std::unique_ptr<kvpool> p(new kvpool);
  p->cuda_device = cuda_device;
  CU(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, cuda_device));
  p->geom = *g;
  p->kvb = kvb;
  p->payload = 2 * kvb;
  p->n = n_devs;
  p->bandwidth = bw;
  p->w = w;
  default_tuning(p.get());
  auto cleanup = [&]() {
    for (auto& b : p->bufs) host_buffer_free(&b);
    for (auto s : p->own_streams) cudaStreamDestroy(s);
    if (p->table_arena) cudaFree(p->table_arena);
    if (p->table_arena_host) cudaFreeHost(p->table_arena_host);
    if (p->upload) cudaStreamDestroy(p->upload);
    if (p->join_out) cudaStreamDestroy(p->join_out);
  };
  p->bufs.resize(n_devs);
  for (uint32_t i = 0; i < n_devs; ++i) {
    std::string err;
    const bool hbm = devs[i].flags & KVPOOL_DEV_HBM;
    const int rc = hbm ? device_buffer_alloc(&p->bufs[i], devs[i].capacity_bytes, devs[i].gpu < 0 ? cuda_device : devs[i].gpu, cuda_device, &err)
                       : host_buffer_alloc(&p->bufs[i], devs[i].capacity_bytes,
                                           devs[i].numa_node == KVPOOL_NUMA_AUTO ? gpu_numa_node(cuda_device) : devs[i].numa_node, devs[i].flags & KVPOOL_DEV_WRITE_COMBINED,
                                           devs[i].flags & KVPOOL_DEV_NUMA_STRICT, devs[i].flags & KVPOOL_DEV_CUDA_HOSTALLOC, &err);
    if (rc == KVPOOL_OK && hbm) p->hbm_mask |= 1u << i;
    if (rc != KVPOOL_OK) {
      cleanup();
      return fail(rc, "create: pool device %u (%llu bytes): %s", i, (unsigned long long)devs[i].capacity_bytes, err.c_str());
    }
    p->alloc.emplace_back(devs[i].capacity_bytes);
  }
  // one I/O stream per direction and per independent resource: a device of its own (link_group 0) gets its own pair, the
  // members of a link group share the pair of the group's first member, so their copies run in the order they were asked for
  p->io.resize(n_devs, nullptr);
  p->io_out.resize(n_devs, nullptr);
  p->link_group.resize(n_devs);
  for (uint32_t i = 0; i < n_devs; ++i) {
    p->link_group[i] = devs[i].link_group;
    uint32_t first = i;
    for (uint32_t j = 0; j < i && devs[i].link_group; ++j)
      if (devs[j].link_group == devs[i].link_group) { first = j; break; }
    if (first != i) { p->io[i] = p->io[first]; p->io_out[i] = p->io_out[first]; continue; }
    for (auto* v : {&p->io, &p->io_out}) {
      cudaError_t e = cudaStreamCreateWithFlags(&(*v)[i], cudaStreamNonBlocking);
      if (e != cudaSuccess) { cleanup(); return fail(KVPOOL_ECUDA, "cudaStreamCreate: %s", cudaGetErrorString(e)); }
      p->own_streams.push_back((*v)[i]);
    }
  }
  if (cudaMalloc(reinterpret_cast<void**>(&p->table_arena), kTableArenaBytes) != cudaSuccess) {
    cudaGetLastError();
    cleanup();
    return fail(KVPOOL_ENOMEM, "create: table arena");
  }
  if (cudaHostAlloc(reinterpret_cast<void**>(&p->table_arena_host), kTableArenaBytes, cudaHostAllocDefault) != cudaSuccess ||
      cudaStreamCreateWithFlags(&p->upload, cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&p->join_out, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    cleanup();
    return fail(KVPOOL_ENOMEM, "create: table arena mirror / upload stream");
  }
  p->table_alloc = StripeAllocator(kTableArenaBytes, 256);
  *out = p.release();
  return KVPOOL_OK;
}

int kvpool_destroy(kvpool_t* p) {
  if (!p) return fail(KVPOOL_EINVAL, "destroy: null pool");
  DeviceGuard guard(p->cuda_device);
  cudaDeviceSynchronize();
  for (auto* pl : p->live) destroy_placement(p, pl);
  p->live.clear();
  free_slots(p);
  for (auto s : p->own_streams) cudaStreamDestroy(s);
  for (auto& b : p->bufs) host_buffer_free(&b);
  if (p->table_arena) cudaFree(p->table_arena);
  if (p->table_arena_host) cudaFreeHost(p->table_arena_host);
  if (p->upload) cudaStreamDestroy(p->upload);
  if (p->join_out) cudaStreamDestroy(p->join_out);
  for (auto& kv : p->prof_side) { cudaStreamDestroy(kv.second.first); cudaStreamDestroy(kv.second.second); }
  for (auto e : p->ev_free) cudaEventDestroy(e);
  for (auto& r : p->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
  for (auto e : p->prof_free) cudaEventDestroy(e);
  if (p->span_arena) cudaFree(p->span_arena);
  if (p->bad_d) cudaFree(p->bad_d);
  delete p;
  return KVPOOL_OK;
}

int kvpool_set_bandwidth(kvpool_t* p, const double* bw) {
  PoolLock lock__(p);
  if (!p || !bw) return fail(KVPOOL_EINVAL, "set_bandwidth: null argument");
  if (!p->live.empty()) return fail(KVPOOL_ESTATE, "set_bandwidth: %zu placements are live", p->live.size());
  std::vector<uint64_t> w(p->n);
  if (!quantise_weights(bw, p->n, w.data())) return fail(KVPOOL_EINVAL, "set_bandwidth: bandwidth must be positive (>= 0.0005 GB/s)");
  p->bandwidth.assign(bw, bw + p->n);
  p->w = w;
  return KVPOOL_OK;
}

int kvpool_measure_bandwidth(kvpool_t* p, uint32_t dev, int direction, uint64_t bytes, uint32_t iters, double* gbps_out) {
  PoolLock lock__(p);
  if (!p || !gbps_out || dev >= p->n || bytes == 0 || iters == 0 || direction < 0 || direction > KVPOOL_MEASURE_KERNEL_OFFLOAD)
    return fail(KVPOOL_EINVAL, "measure_bandwidth: bad arguments");
  if (bytes > p->bufs[dev].bytes) return fail(KVPOOL_EINVAL, "measure_bandwidth: %llu bytes exceed the pool buffer", (unsigned long long)bytes);
  if (!p->live.empty()) return fail(KVPOOL_ESTATE, "measure_bandwidth: %zu placements are live", p->live.size());
  DeviceGuard guard(p->cuda_device);
  void* scratch = nullptr;
  CU(cudaMalloc(&scratch, bytes));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  std::vector<float> ms(iters);
  const bool by_kernel = direction >= KVPOOL_MEASURE_KERNEL_RETRIEVE, towards_gpu = direction == 0 || direction == KVPOOL_MEASURE_KERNEL_RETRIEVE;
  cudaStream_t s = towards_gpu ? p->io[dev] : p->io_out[dev];
  int rc = KVPOOL_OK;
  // kernel modes: K blocks, block u at slot u of the device's buffer and at physical block u of the scratch paged layout
  // (K plane then V plane): one device-major launch whose inverse map and block table are both the identity
  const uint32_t K = static_cast<uint32_t>(std::min<uint64_t>(bytes / p->payload, 0x7fffffffull));
  uint32_t* ident = nullptr;
  LayerArgs ka{};
  if (by_kernel) {
    if (K == 0) { cudaFree(scratch); cudaEventDestroy(e0); cudaEventDestroy(e1); return fail(KVPOOL_EINVAL, "measure_bandwidth: fewer bytes than one KV cache (%llu)", (unsigned long long)p->payload); }
    bytes = static_cast<uint64_t>(K) * p->payload;
    std::vector<uint32_t> h(K);
    std::iota(h.begin(), h.end(), 0u);
    CU(cudaMalloc(reinterpret_cast<void**>(&ident), static_cast<uint64_t>(K) * 4));
    CU(cudaMemcpyAsync(ident, h.data(), static_cast<uint64_t>(K) * 4, cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));
    ka.k_base = static_cast<uint8_t*>(scratch);
    ka.v_base = static_cast<uint8_t*>(scratch) + static_cast<uint64_t>(K) * p->kvb;
    ka.stride = p->kvb;
    ka.table = reinterpret_cast<const int32_t*>(ident);
    ka.order = ident;
    ka.K = K;
    ka.kvb = static_cast<uint32_t>(p->kvb);
    ka.pool_base[0] = reinterpret_cast<uint64_t>(p->bufs[dev].dev_alias);
  }
  if (towards_gpu && !is_hbm(p, dev)) {
    // Pages the CPU has just zeroed sit partly in its caches; host->GPU DMA reads of such lines run 5 % slow until a DMA
    // write has claimed them (measured: 52 -> 55.6 GB/s after one pass).  Stripes are always written by an offload
    // before a retrieve reads them, so that is the state to measure: write the region once (no placement is live).
    CU(cudaMemcpyAsync(pool_bytes(p, dev), scratch, bytes, cudaMemcpyDefault, s));
    p->n_memcpys++;
  }
  for (uint32_t it = 0; it < iters + 1 && rc == KVPOOL_OK; ++it) {  // first pass is a warm-up
    cudaEventRecord(e0, s);
    cudaError_t e;
    if (by_kernel) {
      e = launch_layer_copy(ka, !towards_gpu, launch_cfg(p, !is_hbm(p, dev)), s);
      p->n_kernels++;
    } else {
      e = towards_gpu ? cudaMemcpyAsync(scratch, pool_bytes(p, dev), bytes, cudaMemcpyDefault, s)
                      : cudaMemcpyAsync(pool_bytes(p, dev), scratch, bytes, cudaMemcpyDefault, s);
      p->n_memcpys++;
    }
    cudaEventRecord(e1, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { rc = fail(KVPOOL_ECUDA, "measure_bandwidth: %s", cudaGetErrorString(e)); break; }
    if (it > 0) cudaEventElapsedTime(&ms[it - 1], e0, e1);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(scratch);
  if (ident) cudaFree(ident);
  if (rc != KVPOOL_OK) return rc;
  std::sort(ms.begin(), ms.end());
  *gbps_out = static_cast<double>(bytes) / (ms[iters / 2] * 1.0e6);
  return KVPOOL_OK;
}

int kvpool_share_bandwidth(const double* alone, const uint32_t* link_group, uint32_t n, double* out) {
  if (!alone || !link_group || !out || n == 0 || n > KVPOOL_MAX_DEVICES) return fail(KVPOOL_EINVAL, "share_bandwidth: bad arguments");
  for (uint32_t i = 0; i < n; ++i)
    if (!(alone[i] > 0.0) || !(alone[i] < 1e300)) return fail(KVPOOL_EINVAL, "share_bandwidth: bandwidth %u is not positive and finite", i);
  for (uint32_t i = 0; i < n; ++i) {
    if (link_group[i] == 0) { out[i] = alone[i]; continue; }
    double best = 0.0, sum = 0.0;  // summed in index order
    for (uint32_t j = 0; j < n; ++j)
      if (link_group[j] == link_group[i]) { best = std::max(best, alone[j]); sum += alone[j]; }
    out[i] = alone[i] * best / sum;
  }
  return KVPOOL_OK;
}

int kvpool_calibrate(kvpool_t* p, int direction, uint64_t bytes, uint32_t iters, double* bandwidth_out) {
  PoolLock lock__(p);
  if (!p || bytes == 0 || iters == 0 || direction < 0 || direction > KVPOOL_MEASURE_KERNEL_OFFLOAD) return fail(KVPOOL_EINVAL, "calibrate: bad arguments");
  if (!p->live.empty()) return fail(KVPOOL_ESTATE, "calibrate: %zu placements are live", p->live.size());
  std::vector<double> alone(p->n), shared(p->n);
  for (uint32_t i = 0; i < p->n; ++i) {
    const int rc = kvpool_measure_bandwidth(p, i, direction, std::min<uint64_t>(bytes, p->bufs[i].bytes), iters, &alone[i]);
    if (rc != KVPOOL_OK) return rc;
  }
  int rc = kvpool_share_bandwidth(alone.data(), p->link_group.data(), p->n, shared.data());
  if (rc == KVPOOL_OK) rc = kvpool_set_bandwidth(p, shared.data());
  if (rc != KVPOOL_OK) return rc;
  if (bandwidth_out) std::copy(shared.begin(), shared.end(), bandwidth_out);
  return KVPOOL_OK;
}

int kvpool_bandwidths(const kvpool_t* p, double* bandwidth_out, uint32_t* link_group_out) {
  if (!p) return fail(KVPOOL_EINVAL, "bandwidths: null pool");
  if (bandwidth_out) std::copy(p->bandwidth.begin(), p->bandwidth.end(), bandwidth_out);
  if (link_group_out) std::copy(p->link_group.begin(), p->link_group.end(), link_group_out);
  return KVPOOL_OK;
}

int kvpool_set_path(kvpool_t* p, int path) {
  PoolLock lock__(p);
  if (!p || path < KVPOOL_PATH_AUTO || path > KVPOOL_PATH_HYBRID) return fail(KVPOOL_EINVAL, "set_path: bad arguments");
  p->path = path;
  return KVPOOL_OK;
}

int kvpool_set_tuning(kvpool_t* p, const kvpool_tuning* t) {
  PoolLock lock__(p);
  if (!p || !t) return fail(KVPOOL_EINVAL, "set_tuning: null argument");
  if (t->kernel > KVPOOL_KERNEL_BULK || t->link_kernel > KVPOOL_KERNEL_BULK)
    return fail(KVPOOL_EINVAL, "set_tuning: unknown kernel %u / link_kernel %u", t->kernel, t->link_kernel);
  if (t->bulk_chunk && (t->bulk_chunk < 1024 || t->bulk_chunk > 32768 || (t->bulk_chunk & (t->bulk_chunk - 1))))
    return fail(KVPOOL_EINVAL, "set_tuning: bulk_chunk must be a power of two in 1 KiB..32 KiB");
  if (t->bulk_stages > 8 || t->bulk_stages == 1) return fail(KVPOOL_EINVAL, "set_tuning: bulk_stages must be 2..8");
  if (t->bulk_warps > 8) return fail(KVPOOL_EINVAL, "set_tuning: bulk_warps must be 1..8");
  if (t->stage_slots > 64) return fail(KVPOOL_EINVAL, "set_tuning: stage_slots must be <= 64");
  if (t->vec_threads && (t->vec_threads % 32 || t->vec_threads < 64 || t->vec_threads > 512))
    return fail(KVPOOL_EINVAL, "set_tuning: vec_threads must be a multiple of 32 in 64..512");
  if (t->pdl > 2) return fail(KVPOOL_EINVAL, "set_tuning: pdl must be 0 (keep), 1 (on) or 2 (off)");
  if (t->vec_unroll && t->vec_unroll != 4 && t->vec_unroll != 8 && t->vec_unroll != 16)
    return fail(KVPOOL_EINVAL, "set_tuning: vec_unroll must be 4, 8 or 16");
  kvpool_tuning d = p->tune;
  d.kernel = t->kernel;
  d.link_kernel = t->link_kernel;
  if (t->hbm_ctas) d.hbm_ctas = t->hbm_ctas;
  if (t->link_ctas) d.link_ctas = t->link_ctas;
  if (t->bulk_chunk) d.bulk_chunk = t->bulk_chunk;
  if (t->bulk_stages) d.bulk_stages = t->bulk_stages;
  if (t->bulk_warps) d.bulk_warps = t->bulk_warps;
  if (t->vec_threads) d.vec_threads = t->vec_threads;
  if (t->vec_unroll) d.vec_unroll = t->vec_unroll;
  if (t->pdl) d.pdl = t->pdl;
  if (t->auto_threshold_bytes) d.auto_threshold_bytes = t->auto_threshold_bytes;
  if (t->group_bytes) d.group_bytes = t->group_bytes;
  if (t->stage_chunk_bytes) d.stage_chunk_bytes = t->stage_chunk_bytes == ~0ull ? 0 : t->stage_chunk_bytes;
  if (t->stage_slots && t->stage_slots != d.stage_slots) {
    DeviceGuard guard(p->cuda_device);
    d.stage_slots = t->stage_slots;
    p->tune = d;
    const uint64_t bytes = p->slot_bytes;
    CU(cudaDeviceSynchronize());
    free_slots(p);
    if (bytes) return ensure_slots(p, bytes);
    return KVPOOL_OK;
  }
  p->tune = d;
  return KVPOOL_OK;
}

int kvpool_reserve_staging(kvpool_t* p, uint64_t bytes) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "reserve_staging: null pool");
  if (all_hbm(p)) return KVPOOL_OK;  // nothing is ever staged
  DeviceGuard guard(p->cuda_device);
  return ensure_slots(p, bytes + static_cast<uint64_t>(p->n) * 256 * (kMaxBatch + 1));
}

int kvpool_get_tuning(const kvpool_t* p, kvpool_tuning* t_out) {
  if (!p || !t_out) return fail(KVPOOL_EINVAL, "get_tuning: null argument");
  *t_out = p->tune;
  return KVPOOL_OK;
}

int kvpool_place(kvpool_t* p, const uint32_t* blocks_per_layer, kvpool_placement_t** out) {
  if (!p || !blocks_per_layer || !out) return fail(KVPOOL_EINVAL, "place: null argument");
  *out = nullptr;
  std::lock_guard<std::recursive_mutex> lock(p->mu);
  DeviceGuard guard(p->cuda_device);
  const uint32_t L = p->geom.n_layers, N = p->n;
  std::unique_ptr<kvpool_placement> pl(new kvpool_placement);
  pl->pool = p;
  pl->layers.resize(L);

  // a1-a3: counts and weighted round-robin, once per distinct K (layers of equal size share their map)
  std::unordered_map<uint64_t, std::shared_ptr<LayerMap>> by_k;
  uint64_t table_bytes = 0, max_layer_bytes = 0;
  for (uint32_t l = 0; l < L; ++l) {
    const uint64_t K = blocks_per_layer[l];
    auto it = by_k.find(K);
    if (it == by_k.end()) {
      auto m = std::make_shared<LayerMap>();
      m->K = K;
      m->counts.resize(N);
      m->start.resize(N);
      m->dev.resize(K);
      m->slot.resize(K);
      target_counts(p->w.data(), N, K, m->counts.data());
      wrr_closed_form(m->counts.data(), N, K, m->dev.data(), m->slot.data());
      uint32_t acc = 0;
      for (uint32_t i = 0; i < N; ++i) { m->start[i] = acc; acc += m->counts[i]; }
      m->order.resize(K);
      for (uint64_t j = 0; j < K; ++j) m->order[m->start[m->dev[j]] + m->slot[j]] = static_cast<uint32_t>(j);
      for (uint32_t i = 0; i < N; ++i)
        if (!is_hbm(p, i)) m->host_blocks += m->counts[i];
      table_bytes += (2 + (p->hbm_mask && !all_hbm(p) ? 1 : 0)) * ((K * 4 + 255) / 256 * 256) + (K + 255) / 256 * 256;
      it = by_k.emplace(K, std::move(m)).first;
    }
    pl->layers[l].map = it->second;
    max_layer_bytes = std::max(max_layer_bytes, K * p->payload);
  }

  const uint64_t bases_bytes = (static_cast<uint64_t>(L) * N * 8 + 255) / 256 * 256;
  table_bytes += bases_bytes;

  // a4: stripe allocation, all or nothing.  Each pool device gets ONE contiguous region per placement in which the
  // layers' stripes follow each other in layer order (256-byte aligned), so that a run of consecutive layers is also
  // one contiguous span per device — what lets the batched calls move several small layers with one copy per device.
  constexpr uint64_t kStripeAlign = 256;
  pl->region_off.assign(N, 0);
  pl->region_bytes.assign(N, 0);
  for (uint32_t l = 0; l < L; ++l) {
    auto& Ls = pl->layers[l];
    Ls.stripe_off.assign(N, 0);
    for (uint32_t i = 0; i < N; ++i) {
      Ls.stripe_off[i] = pl->region_bytes[i];  // relative for now
      pl->region_bytes[i] += (static_cast<uint64_t>(Ls.map->counts[i]) * p->payload + kStripeAlign - 1) / kStripeAlign * kStripeAlign;
    }
  }
  bool ok = true;
  uint32_t fail_dev = 0, done_devs = 0;
  for (uint32_t i = 0; i < N; ++i) {
    if (!p->alloc[i].alloc(pl->region_bytes[i], &pl->region_off[i])) { ok = false; fail_dev = i; break; }
    done_devs = i + 1;
  }
  auto rollback = [&]() {
    for (uint32_t i = 0; i < done_devs; ++i) p->alloc[i].free(pl->region_off[i], pl->region_bytes[i]);
    pl->region_off.clear();
    free_tables(p, pl.get());
    for (auto& Ls : pl->layers)
      if (Ls.landed) p->ev_free.push_back(Ls.landed);
  };
  if (!ok) {
    rollback();
    return fail(KVPOOL_ENOMEM, "place: pool device %u has no contiguous %llu bytes (capacity %llu, used %llu)", fail_dev,
                (unsigned long long)pl->region_bytes[fail_dev], (unsigned long long)p->alloc[fail_dev].capacity(),
                (unsigned long long)p->alloc[fail_dev].used());
  }
  for (auto& Ls : pl->layers)
    for (uint32_t i = 0; i < N; ++i) Ls.stripe_off[i] += pl->region_off[i];

  // GLT upload: dense (device_id, slot) columns, one device allocation per placement
  if (table_bytes) {
    cudaError_t e = cudaSuccess;
    uint64_t arena_off = 0;
    pl->tables_bytes = table_bytes;
    if (p->table_alloc.alloc(table_bytes, &arena_off)) {
      pl->tables_d = p->table_arena + arena_off;
      pl->tables_in_arena = true;
    } else {
      e = cudaMalloc(reinterpret_cast<void**>(&pl->tables_d), table_bytes);  // arena exhausted: private allocation
      if (e != cudaSuccess) { cudaGetLastError(); pl->tables_d = nullptr; rollback(); return fail(KVPOOL_ENOMEM, "place: table upload buffer: %s", cudaGetErrorString(e)); }
    }
    // built in the pinned mirror of the arena (or, for a private allocation, in pageable memory) and uploaded on the
    // library's own stream: no use of the legacy default stream, so no implicit wait for the application's work
    std::vector<uint8_t> pageable(pl->tables_in_arena ? 0 : table_bytes);
    uint8_t* const host = pl->tables_in_arena ? p->table_arena_host + arena_off : pageable.data();
    uint64_t off = 0;
    for (auto& kv : by_k) {
      LayerMap& m = *kv.second;
      if (m.K == 0) continue;
      m.slot_d = reinterpret_cast<const uint32_t*>(pl->tables_d + off);
      memcpy(host + off, m.slot.data(), m.K * 4);
      off += (m.K * 4 + 255) / 256 * 256;
      m.order_d = reinterpret_cast<const uint32_t*>(pl->tables_d + off);  // per-device inverse map, for device-major chunks
      memcpy(host + off, m.order.data(), m.K * 4);
      off += (m.K * 4 + 255) / 256 * 256;
      m.dev_d = pl->tables_d + off;
      memcpy(host + off, m.dev.data(), m.K);
      off += (m.K + 255) / 256 * 256;
      if (p->hbm_mask && !all_hbm(p)) {  // visiting order: host-device blocks first, each class in logical order
        uint32_t* v = reinterpret_cast<uint32_t*>(host + off);
        uint64_t at = 0;
        for (int hbm_pass = 0; hbm_pass < 2; ++hbm_pass)
          for (uint64_t j = 0; j < m.K; ++j)
            if (is_hbm(p, m.dev[j]) == (hbm_pass == 1)) v[at++] = static_cast<uint32_t>(j);
        m.visit_d = reinterpret_cast<const uint32_t*>(pl->tables_d + off);
        off += (m.K * 4 + 255) / 256 * 256;
      }
    }
    for (uint32_t l = 0; l < L; ++l) {  // GPU-visible stripe addresses, one row per layer
      uint64_t* row = reinterpret_cast<uint64_t*>(host + off) + static_cast<uint64_t>(l) * N;
      for (uint32_t i = 0; i < N; ++i)
        row[i] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(p->bufs[i].dev_alias) + pl->layers[l].stripe_off[i]);
      pl->layers[l].base_d = reinterpret_cast<const uint64_t*>(pl->tables_d + off) + static_cast<uint64_t>(l) * N;
    }
    off += bases_bytes;
    e = cudaMemcpyAsync(pl->tables_d, host, off, cudaMemcpyHostToDevice, p->upload);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->upload);  // the tables are in place before any launch can name them
    if (e != cudaSuccess) { rollback(); return fail(KVPOOL_ECUDA, "place: table upload: %s", cudaGetErrorString(e)); }
  }
  for (auto& Ls : pl->layers) {
    cudaError_t e = take_event(p, &Ls.landed);
    if (e != cudaSuccess) { rollback(); return fail(KVPOOL_ECUDA, "place: cudaEventCreate: %s", cudaGetErrorString(e)); }
  }
  if (p->path != KVPOOL_PATH_ZEROCOPY && !all_hbm(p)) {
    // a slot holds the largest layer, or a group of small layers (plus the 256-byte alignment gaps between stripes)
    const uint64_t total_bytes = std::accumulate(pl->region_bytes.begin(), pl->region_bytes.end(), uint64_t{0});
    const uint64_t group_cap = std::min<uint64_t>(std::max<uint64_t>(max_layer_bytes, p->tune.group_bytes), total_bytes);
    uint64_t want = std::max(max_layer_bytes, group_cap);
    if (p->tune.stage_chunk_bytes) want = std::min(want, std::max<uint64_t>(p->tune.stage_chunk_bytes, p->payload));  // larger layers travel in chunks
    const int rc = ensure_slots(p, want + static_cast<uint64_t>(N) * 256 * (kMaxBatch + 1));
    if (rc != KVPOOL_OK) { rollback(); return rc; }
  }
  p->live.push_back(pl.get());
  *out = pl.release();
  return KVPOOL_OK;
}

int kvpool_release(kvpool_t* p, kvpool_placement_t* pl) {
  if (!p || !pl) return fail(KVPOOL_EINVAL, "release: null argument");
  std::lock_guard<std::recursive_mutex> lock(p->mu);
  auto it = std::find(p->live.begin(), p->live.end(), pl);
  if (it == p->live.end()) return fail(KVPOOL_EINVAL, "release: placement does not belong to this pool");
  DeviceGuard guard(p->cuda_device);
  const int rc = sync_pool_streams(p);  // the library's own transfers for it must be over
  if (rc != KVPOOL_OK) return rc;
  for (auto& u : pl->last_use) CU(cudaEventSynchronize(u.second));  // and so must the kernels it put on the caller's streams
  p->live.erase(it);
  destroy_placement(p, pl);
  return KVPOOL_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------
// hot path
// ---------------------------------------------------------------------------------------------------
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
  bool host_blocks = false, hbm_blocks = false;
};
static ChunkPlan plan_chunk(const kvpool* p, const LayerState& L, uint32_t first, uint32_t n) {
  ChunkPlan c;
  uint64_t acc = 0;
  for (uint32_t i = 0; i < p->n; ++i) {
    slot_range(*L.map, i, first, n, &c.lo[i], &c.hi[i]);
    c.off[i] = acc;
    if (c.hi[i] == c.lo[i]) continue;
    if (is_hbm(p, i)) { c.hbm_blocks = true; continue; }
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
  if (per_slot == 0) return fail(KVPOOL_ESTATE, "offload: no staging slot (the placement was made while the path was zero-copy)");
  // `landed` must mean "all stripes complete": it is recorded on a stream of the pool's own that carries no copies and only
  // gathers every chunk's kernel and copies — the per-device I/O streams never wait for one another
  cudaStream_t lead = p->join_out;
  if (L.landed_pending) CU(cudaStreamWaitEvent(lead, L.landed, 0));  // `landed` keeps covering what was offloaded before
  // an earlier offload of this layer may still be writing the HBM-type stripes the kernel stores into
  if (whole.hbm_blocks && L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
  if (n_blocks > per_slot) {
    // DEVICE-MAJOR chunks: a chunk is a run of consecutive slots of one device's stripe, gathered by a launch that finds its
    // logical blocks through that device's inverse map, and leaves the slot as ONE copy.  An HBM-type device's share is
    // gathered in place by one launch.
    a.order = L.map->order_d;
    for (uint32_t i = 0; i < N; ++i) {
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
  if (per_slot == 0) return fail(KVPOOL_ESTATE, "retrieve: no staging slot (the placement was made while the path was zero-copy)");
  if (whole.hbm_blocks && L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));  // HBM-type stripes are read in place
  if (n_blocks > per_slot) {
    // DEVICE-MAJOR chunks (see kvpool_offload_range): one copy fills a slot with a run of one device's slots, one launch
    // scatters them through that device's inverse map; the copy of the next chunk overlaps it
    a.order = L.map->order_d;
    for (uint32_t i = 0; i < N; ++i) {
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

// One multi-layer launch, counted and (when profiling) bracketed by an event pair on `s`.
static int launch_multi_counted(kvpool* p, const MultiArgs& ma, bool pack, bool link_bound, cudaStream_t s) {
  ProfRec r;
  if (p->profiling) {
    r.bytes = static_cast<uint64_t>(ma.total_units) * p->payload;
    r.kind = (link_bound ? 2 : 0) + (pack ? 0 : 1);
    const int rc = prof_begin(p, &r, s);
    if (rc != KVPOOL_OK) return rc;
  }
  MultiArgs timed = ma;
  if (p->profiling) timed.span = take_span(p, &r);
  CU(launch_multi_copy(timed, pack, launch_cfg(p, link_bound, pack), s));
  p->n_kernels++;
  if (p->profiling) return prof_end(p, &r, s);
  return KVPOOL_OK;
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
};

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
  for (uint32_t b = 0; b < g.n; ++b) {
    LayerState& L = c.pl->layers[c.first + g.q[b]];
    if (L.landed_pending) CU(cudaStreamWaitEvent(c.s, L.landed, 0));  // settled (no wait) after kvpool_synchronize
  }
  const int rc = launch_multi_counted(p, ma, c.pack, true, c.s);
  if (rc != KVPOOL_OK) return rc;
  if (c.pack)
    for (uint32_t b = 0; b < g.n; ++b) {
      LayerState& L = c.pl->layers[c.first + g.q[b]];
      L.offloaded = true;
      L.have.clear();
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
  const int rc = issue_group_work(c, g);
  if (rc != KVPOOL_OK || !c.ready) return rc;
  for (uint32_t b = 0; b < g.n; ++b)
    if (c.ready[g.q[b]]) CU(cudaEventRecord(static_cast<cudaEvent_t>(c.ready[g.q[b]]), c.s));
  return KVPOOL_OK;
}

int issue_group_work(const BatchCall& c, const LayerGroup& g) {
  kvpool* p = c.p;
  if (!use_staged(p, c.pack, g.host_bytes)) return issue_zero_copy_group(c, g);
  if (g.n > 1) {
    const int rc = issue_staged_group(c, g);
    if (rc != 1) return rc;
  }
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
static int layers_batched(kvpool_t* p, kvpool_placement_t* pl, bool pack, uint32_t first, uint32_t n, const void* const* k_bases,
                          const void* const* v_bases, uint64_t stride, const int32_t* const* tables, void* cuda_stream,
                          void* const* ready = nullptr) {
  PoolLock lock__(p);
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
  const BatchCall c{p, pl, pack, first, k_bases, v_bases, tables, stride, static_cast<cudaStream_t>(cuda_stream), ready};
  uint64_t cap = std::max<uint64_t>(p->tune.group_bytes, 1);
  if (ready) {
    // a consumer follows behind the per-layer events: a request so small that it would travel as ONE group (all layers
    // ready together, the consumer not overlapped at all) is cut in two, so that the consumer of the first half runs
    // under the transfer of the second (GPT-OSS-shaped KV at 1K context: 27 MiB; profiles/r2_blocked_io.txt)
    uint64_t total = 0;
    for (uint32_t q = 0; q < n; ++q) total += pl->layers[first + q].map->K * p->payload;
    if (total < cap) cap = std::max<uint64_t>((total + 1) / 2, 1);
  }
  LayerGroup g;
  uint64_t units = 0;
  for (uint32_t q = 0; q < n; ++q) {
    LayerState& L = pl->layers[first + q];
    if (L.map->K == 0) {  // nothing to move: ready in stream order right away
      if (pack) L.offloaded = true;
      if (ready && ready[q]) CU(cudaEventRecord(static_cast<cudaEvent_t>(ready[q]), c.s));
      continue;
    }
    const uint64_t bytes = L.map->K * p->payload;
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
  const int rc = issue_group(c, g);
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

// Baseline for comparison: 2*K_l individual cudaMemcpyAsync calls per layer, no kernel.
static int naive_layer(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, bool pack, const void* k_base, const void* v_base, uint64_t stride,
                       const int32_t* table_host, void* cuda_stream) {
  PoolLock lock__(p);
  int rc = check_layer_call(p, pl, layer, k_base, v_base, stride, table_host);
  if (rc != KVPOOL_OK) return rc;
  LayerState& L = pl->layers[layer];
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
  for (auto& L : pl->layers)
    if (L.landed_pending) CU(cudaStreamWaitEvent(s, L.landed, 0));
  return KVPOOL_OK;
}

int kvpool_synchronize(kvpool_t* p) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "synchronize: null pool");
  DeviceGuard guard(p->cuda_device);
  const int rc = sync_pool_streams(p);
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

int kvpool_spin(kvpool_t* p, uint64_t ns, void* cuda_stream) {
  PoolLock lock__(p);
  if (!p) return fail(KVPOOL_EINVAL, "spin: null pool");
  if (ns > 10ull * 1000 * 1000 * 1000) return fail(KVPOOL_EINVAL, "spin: more than 10 s");
  DeviceGuard guard(p->cuda_device);
  CU(launch_spin(ns, static_cast<cudaStream_t>(cuda_stream)));
  p->n_kernels++;
  return KVPOOL_OK;
}

// ---------------------------------------------------------------------------------------------------
// introspection
// ---------------------------------------------------------------------------------------------------
int kvpool_n_devices(const kvpool_t* p, uint32_t* n_out) {
  if (!p || !n_out) return fail(KVPOOL_EINVAL, "n_devices: null argument");
  *n_out = p->n;
  return KVPOOL_OK;
}

int kvpool_weights(const kvpool_t* p, uint64_t* w_out) {
  if (!p || !w_out) return fail(KVPOOL_EINVAL, "weights: null argument");
  std::copy(p->w.begin(), p->w.end(), w_out);
  return KVPOOL_OK;
}

int kvpool_device_info(const kvpool_t* p, uint32_t dev, void** host_base, uint64_t* capacity, uint64_t* used, int32_t* numa_actual) {
  if (!p || dev >= p->n) return fail(KVPOOL_EINVAL, "device_info: bad arguments");
  if (host_base) *host_base = p->bufs[dev].host;
  if (capacity) *capacity = p->bufs[dev].bytes;
  if (used) *used = p->alloc[dev].used();
  if (numa_actual) *numa_actual = p->bufs[dev].numa_actual;
  return KVPOOL_OK;
}

int kvpool_counts(const kvpool_placement_t* pl, uint32_t layer, uint32_t* counts_out) {
  if (!pl || !counts_out || layer >= pl->layers.size()) return fail(KVPOOL_EINVAL, "counts: bad arguments");
  const auto& c = pl->layers[layer].map->counts;
  std::copy(c.begin(), c.end(), counts_out);
  return KVPOOL_OK;
}

int kvpool_lookup(const kvpool_placement_t* pl, uint32_t layer, uint32_t block, uint32_t* device_id, uint32_t* type, uint32_t* slot,
                  void** host_ptr) {
  if (!pl || layer >= pl->layers.size()) return fail(KVPOOL_EINVAL, "lookup: bad arguments");
  const LayerState& L = pl->layers[layer];
  if (block >= L.map->K) return fail(KVPOOL_EINVAL, "lookup: block %u out of range (K %llu)", block, (unsigned long long)L.map->K);
  const uint32_t d = L.map->dev[block], s = L.map->slot[block];
  if (device_id) *device_id = d;
  if (type) *type = is_hbm(pl->pool, d) ? KVPOOL_TYPE_HBM : KVPOOL_TYPE_MEM;
  if (slot) *slot = s;
  if (host_ptr) *host_ptr = pool_bytes(pl->pool, d) + L.stripe_off[d] + static_cast<uint64_t>(s) * pl->pool->payload;
  return KVPOOL_OK;
}

int kvpool_stripe(const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, void** host_ptr, uint64_t* nbytes) {
  if (!pl || layer >= pl->layers.size() || dev >= pl->pool->n) return fail(KVPOOL_EINVAL, "stripe: bad arguments");
  const LayerState& L = pl->layers[layer];
  const uint64_t bytes = static_cast<uint64_t>(L.map->counts[dev]) * pl->pool->payload;
  if (host_ptr) *host_ptr = bytes ? pool_bytes(pl->pool, dev) + L.stripe_off[dev] : nullptr;
  if (nbytes) *nbytes = bytes;
  return KVPOOL_OK;
}

int kvpool_stripe_read(kvpool_t* p, const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, void* dst_host, uint64_t nbytes) {
  PoolLock lock__(p);
  if (!p || !pl || pl->pool != p || !is_live(p, pl) || layer >= pl->layers.size() || dev >= p->n) return fail(KVPOOL_EINVAL, "stripe_read: bad arguments");
  const LayerState& L = pl->layers[layer];
  const uint64_t bytes = static_cast<uint64_t>(L.map->counts[dev]) * p->payload;
  if (nbytes > bytes) return fail(KVPOOL_EINVAL, "stripe_read: %llu bytes exceed the stripe's %llu", (unsigned long long)nbytes, (unsigned long long)bytes);
  if (nbytes == 0) return KVPOOL_OK;
  if (!dst_host) return fail(KVPOOL_EINVAL, "stripe_read: null destination");
  const uint8_t* src = pool_bytes(p, dev) + L.stripe_off[dev];
  if (is_hbm(p, dev)) {
    DeviceGuard guard(p->cuda_device);
    CU(cudaMemcpyAsync(dst_host, src, nbytes, cudaMemcpyDeviceToHost, p->upload));
    CU(cudaStreamSynchronize(p->upload));
  } else {
    memcpy(dst_host, src, nbytes);
  }
  return KVPOOL_OK;
}

int kvpool_device_type(const kvpool_t* p, uint32_t dev, uint32_t* type, int32_t* gpu) {
  if (!p || dev >= p->n) return fail(KVPOOL_EINVAL, "device_type: bad arguments");
  if (type) *type = is_hbm(p, dev) ? KVPOOL_TYPE_HBM : KVPOOL_TYPE_MEM;
  if (gpu) *gpu = p->bufs[dev].gpu;
  return KVPOOL_OK;
}

int kvpool_glt_bind(kvpool_t* p, kvpool_placement_t* pl, uint32_t layer, const uint64_t* ids) {
  if (!p || !pl || pl->pool != p || !is_live(p, pl)) return fail(KVPOOL_EINVAL, "glt_bind: bad pool or placement");
  if (layer >= pl->layers.size()) return fail(KVPOOL_EINVAL, "glt_bind: layer %u out of range", layer);
  const uint64_t K = pl->layers[layer].map->K;
  if (K == 0) return KVPOOL_OK;
  if (!ids) return fail(KVPOOL_EINVAL, "glt_bind: null ids");
  std::lock_guard<std::recursive_mutex> lock(p->mu);
  std::unordered_map<uint64_t, GltRef, GltHash> fresh;
  fresh.reserve(K);
  for (uint64_t j = 0; j < K; ++j) {
    if (p->glt.count(ids[j])) return fail(KVPOOL_EINVAL, "glt_bind: identifier 0x%llx is already bound", (unsigned long long)ids[j]);
    if (!fresh.emplace(ids[j], GltRef{pl, layer, static_cast<uint32_t>(j)}).second)
      return fail(KVPOOL_EINVAL, "glt_bind: identifier 0x%llx repeats", (unsigned long long)ids[j]);
  }
  p->glt.insert(fresh.begin(), fresh.end());
  pl->bound_ids.insert(pl->bound_ids.end(), ids, ids + K);
  return KVPOOL_OK;
}

int kvpool_glt_find(kvpool_t* p, uint64_t id, uint64_t* key, uint32_t* device_id, uint32_t* type, void** location, kvpool_placement_t** pl,
                    uint32_t* layer, uint32_t* block) {
  if (!p) return fail(KVPOOL_EINVAL, "glt_find: null pool");
  std::lock_guard<std::recursive_mutex> lock(p->mu);
  const auto it = p->glt.find(id);
  if (it == p->glt.end()) return fail(KVPOOL_ENOENT, "glt_find: identifier 0x%llx is not in the table", (unsigned long long)id);
  const GltRef& r = it->second;
  if (key) *key = GltHash::mix(id);
  if (pl) *pl = r.pl;
  if (layer) *layer = r.layer;
  if (block) *block = r.block;
  return kvpool_lookup(r.pl, r.layer, r.block, device_id, type, nullptr, location);
}

int kvpool_layer_map(const kvpool_placement_t* pl, uint32_t layer, uint8_t* dev_out, uint32_t* slot_out) {
  if (!pl || layer >= pl->layers.size()) return fail(KVPOOL_EINVAL, "layer_map: bad arguments");
  const LayerMap& m = *pl->layers[layer].map;
  if (dev_out) std::copy(m.dev.begin(), m.dev.end(), dev_out);
  if (slot_out) std::copy(m.slot.begin(), m.slot.end(), slot_out);
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

int kvpool_set_table_check(kvpool_t* p, uint64_t nphys) {
  PoolLock lock__(p);
  if (!p || nphys > 0x7fffffffull) return fail(KVPOOL_EINVAL, "set_table_check: null pool or nphys above 2^31-1");
  DeviceGuard guard(p->cuda_device);
  if (nphys && !p->bad_d) {
    CU(cudaMalloc(reinterpret_cast<void**>(&p->bad_d), sizeof(unsigned long long)));
    CU(cudaMemsetAsync(p->bad_d, 0, sizeof(unsigned long long), p->upload));
    CU(cudaStreamSynchronize(p->upload));
  }
  p->check_nphys = static_cast<uint32_t>(nphys);
  return KVPOOL_OK;
}

int kvpool_table_errors(kvpool_t* p, uint64_t* count_out) {
  PoolLock lock__(p);
  if (!p || !count_out) return fail(KVPOOL_EINVAL, "table_errors: null argument");
  *count_out = 0;
  if (!p->bad_d) return KVPOOL_OK;
  DeviceGuard guard(p->cuda_device);
  unsigned long long v = 0;
  CU(cudaMemcpyAsync(&v, p->bad_d, sizeof(v), cudaMemcpyDeviceToHost, p->upload));
  CU(cudaMemsetAsync(p->bad_d, 0, sizeof(v), p->upload));
  CU(cudaStreamSynchronize(p->upload));
  *count_out = v;
  return KVPOOL_OK;
}

int kvpool_stats(const kvpool_t* p, uint64_t* kernel_launches, uint64_t* memcpy_calls) {
  if (!p) return fail(KVPOOL_EINVAL, "stats: null pool");
  if (kernel_launches) *kernel_launches = p->n_kernels;
  if (memcpy_calls) *memcpy_calls = p->n_memcpys;
  return KVPOOL_OK;
}

}  // extern "C"
