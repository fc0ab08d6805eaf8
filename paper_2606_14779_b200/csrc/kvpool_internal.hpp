// Internals shared by the translation units of libkvpool.so: the pool and placement objects behind the opaque handles of
// include/kvpool.h, and the helpers the life-cycle code (kvpool_core.cu), the hot path (kvpool_xfer.cu) and the development
// entry points (kvpool_dev.cu) have in common.  Not installed, not part of the ABI.
#pragma once
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
#include "ssd_io.hpp"

static_assert(KVPOOL_MAX_DEVICES == kvp::kMaxDevices && KVPOOL_MAX_DEVICES == kvp::kMaxDev, "device limit mismatch");

struct kvpool;
struct kvpool_placement;

namespace kvp {

// Sets the calling thread's kvpool_last_error() message and returns `code`.
int fail(int code, const char* fmt, ...);
const char* last_error_message();

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
  // SSD-type devices: ssd_lane_use[i][k] = the latest use of offload lane k of device i that carried a store command of this
  // layer (0 = none; bit i of ssd_stored says there is one).  A stripe larger than a lane is several commands on several
  // lanes, instalments (kvpool_offload_range) add more, and the worker reaps completions in any order: the layer's stripe is
  // on the device once EVERY such lane's cpu_seq flag has reached its entry (uses of one lane complete in order).  The
  // completion is the worker's flag, not an event
  uint32_t ssd_stored = 0;
  std::vector<std::vector<uint32_t>> ssd_lane_use;
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

// One store / retrieve command in flight on an SSD-type device: pinned, GPU-mapped bounce memory — the disk's DMA target on
// one side, read / written by the pack / unpack kernel over the link on the other.
struct SsdLane {
  uint8_t* bounce = nullptr;          // CPU address (the worker's pread / pwrite buffer)
  uint8_t* bounce_dev = nullptr;      // the GPU's address of the same bytes
  uint32_t uses = 0;                  // sequence number of the lane's latest use (the value its flags are compared with)
};
struct SsdState {  // one SSD-type pool device (KV-passthrough)
  SsdDevice io;
  uint8_t* bounce_base = nullptr;  // pinned + mapped host memory: [direction][lane] x lane_bytes
  uint32_t* flags = nullptr;       // pinned + mapped: per direction and lane, gpu_seq (written by a stream write-value, polled
  uint64_t flags_dev = 0;          // by the worker) and cpu_seq (written by the worker, awaited by a stream wait-value)
  uint64_t lane_bytes = 0;
  uint32_t n_lanes = 0;
  std::vector<SsdLane> lane[2];    // [0] retrieve (SSD -> GPU), [1] offload (GPU -> SSD)
  uint32_t cursor[2] = {0, 0};
  // The device's pack / unpack launches run on streams of its own, forked from and joined back to the caller's stream: a
  // launch that waits for a lane (i.e. for the disk) must not hold up the faster devices' launches queued behind it
  cudaStream_t kstream[2] = {nullptr, nullptr};
  cudaEvent_t fork[2] = {nullptr, nullptr}, join[2] = {nullptr, nullptr};
  bool join_pending = false;       // a batched offload joins its pack launches once, at the end of the call
  uint8_t* scratch = nullptr;      // aligned host memory for kvpool_stripe_read / kvpool_measure_bandwidth
};
constexpr uint64_t kSsdScratchBytes = 4ull << 20;

// Per-layer completion flags of one signalled multi-layer retrieve (kernels.cuh, MultiArgs::sig_flag) and the stream that
// turns them into the caller's per-layer events: [wait-value(flag of layer 0)] [record ready[0]] [wait-value(flag 1)] ...
struct SignalSet {
  uint32_t* mem_d = nullptr;       // device: kMaxBatch piece counters, then kMaxBatch flags
  cudaStream_t stream = nullptr;   // a stream per set: a launch held up on its own stream delays nobody else's events
  cudaEvent_t done = nullptr;      // the launch that used the set last has completed (its counters are back at zero)
  uint32_t seq = 0;                // flags of the set's latest launch read >= seq
};
constexpr uint32_t kSignalSets = 8;

}  // namespace kvp

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
  std::vector<kvp::LayerState> layers;
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
  std::vector<kvp::HostBuffer> bufs;
  std::vector<uint32_t> link_group;  // [N] kvpool_device_desc.link_group: devices of one group share io / io_out streams
  std::vector<cudaStream_t> own_streams;  // every stream created for io / io_out, once (members of a group alias one)
  std::vector<kvp::SignalSet> sig;  // made on first use
  uint32_t sig_cursor = 0;
  bool ssd_defer_join = false;  // inside kvpool_offload_layers: see SsdState::join_pending
  uint32_t ssd_mask = 0;  // bit i: pool device i is block storage (KVPOOL_DEV_SSD): its share of a layer moves through bounce lanes
  std::vector<std::unique_ptr<kvp::SsdState>> ssd;  // [N], null for the other types
  uint32_t hbm_mask = 0;  // bit i: pool device i is GPU memory (KVPOOL_DEV_HBM): reached by the kernels directly, never staged or copied
  std::vector<kvp::StripeAllocator> alloc;
  std::vector<cudaStream_t> io;      // one I/O stream per pool device ("independent I/O streams"): host -> GPU copies
  cudaStream_t join_out = nullptr;   // gathers an offload's copies for its `landed` event; carries no work of its own
  std::vector<cudaStream_t> io_out;  // and one for GPU -> host copies, so that an offload and a retrieve use both directions of the link at once
  std::vector<kvp::StageSlot> slots;
  uint64_t slot_bytes = 0;
  uint64_t slot_cursor = 0;
  uint8_t* table_arena = nullptr;  // device memory for placements' GLT columns: no cudaMalloc/cudaFree per request
  uint8_t* table_arena_host = nullptr;  // its pinned host mirror: tables are built in place and uploaded on `upload`
  cudaStream_t upload = nullptr;   // the library's own non-blocking stream for table uploads and small read-backs, so that
                                   // kvpool_place never touches the legacy default stream (which would make it wait for
                                   // whatever the application has queued there)
  kvp::StripeAllocator table_alloc;
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
  std::vector<kvp::ProfRec> prof;
  std::vector<cudaEvent_t> prof_free;  // timing events ready for reuse
  unsigned long long* span_arena = nullptr;  // device: kSpanCap x {min start, max end} in %globaltimer ns, written by the kernels
  uint32_t span_cursor = 0;
  std::recursive_mutex mu;  // every entry point that touches pool state holds it: calls only enqueue work, so the lock is short
};

namespace kvp {

void default_tuning(kvpool* p);
void free_slots(kvpool* p);
int sync_pool_streams(kvpool* p);
int ensure_slots(kvpool* p, uint64_t bytes);  // (re)build the staging ring so that every slot holds `bytes`
bool is_live(const kvpool* p, const kvpool_placement* pl);
void free_tables(kvpool* p, kvpool_placement* pl);
cudaError_t take_event(kvpool* p, cudaEvent_t* e);  // a recycled (or new) cudaEventDisableTiming event
int note_use(kvpool* p, kvpool_placement* pl, cudaStream_t s);
void destroy_placement(kvpool* p, kvpool_placement* pl);
int check_layer_call(kvpool* p, kvpool_placement* pl, uint32_t layer, const void* k_base, const void* v_base, uint64_t stride,
                     const int32_t* table);
LayerArgs base_args(const kvpool* p, const LayerState& L, const void* k_base, const void* v_base, uint64_t stride, const int32_t* table);
LaunchCfg launch_cfg(const kvpool* p, bool link_bound, bool pack = false, bool lane = false);
bool use_staged(const kvpool* p, bool pack, uint64_t host_bytes);
int wait_slot_free(kvpool* p, StageSlot& slot, cudaStream_t s);
void settle_landed(LayerState& L);
// kvpool_dev.cu: launches counted for kvpool_stats and, while profiling is on, bracketed by an event pair and a device-clock span
int launch_counted(kvpool* p, const LayerArgs& a, bool pack, bool link_bound, cudaStream_t s, bool lane = false);
int launch_multi_counted(kvpool* p, const MultiArgs& ma, bool pack, bool link_bound, cudaStream_t s);

// The layer's block table on the device: the caller's, or (null) the one kvpool_set_tables uploaded.
inline const int32_t* table_of(const kvpool_placement* pl, uint32_t layer, const int32_t* given) {
  return given ? given : pl->own_tables_d + pl->own_table_off[layer];
}
inline bool is_hbm(const kvpool* p, uint32_t i) { return (p->hbm_mask >> i) & 1u; }
// Where the CPU / copy engines find pool device i's bytes: the host address, or the device pointer of an HBM device.
inline uint8_t* pool_bytes(const kvpool* p, uint32_t i) {
  return static_cast<uint8_t*>(is_hbm(p, i) ? p->bufs[i].dev_alias : p->bufs[i].host);
}
inline bool is_ssd(const kvpool* p, uint32_t i) { return (p->ssd_mask >> i) & 1u; }
inline bool is_mem(const kvpool* p, uint32_t i) { return !is_hbm(p, i) && !is_ssd(p, i); }
inline bool has_mem(const kvpool* p) { return ((p->hbm_mask | p->ssd_mask) & (p->n >= 32 ? 0xFFFFFFFFu : (1u << p->n) - 1u)) != (p->n >= 32 ? 0xFFFFFFFFu : (1u << p->n) - 1u); }
// kvpool_ssd.cu: stream memory operations (cuStreamWaitValue32 / cuStreamWriteValue32 through the runtime's entry-point query)
int memops_init();                                                        // ECUDA where the driver has none
int stream_wait_geq(cudaStream_t s, uint64_t dev_addr, uint32_t value);  // `s` waits until (int32)(*addr - value) >= 0
int stream_write(cudaStream_t s, uint64_t dev_addr, uint32_t value);     // fenced: earlier writes of `s` are visible first
// kvpool_ssd.cu: SSD-type pool devices
int ssd_open(kvpool* p, uint32_t i, const kvpool_device_desc& d);  // kvpool_create
void ssd_close_all(kvpool* p);                                      // kvpool_destroy / failed create
int ssd_ensure_lanes(kvpool* p);                                    // kvpool_place: bounce lanes, staging pieces, flags, workers
// slots [lo, hi) of layer L's stripe on SSD device i, offload (pack) or retrieve, in lane-sized commands; `a` carries the
// paged side of the launch (bases, stride, table)
int ssd_move(kvpool* p, LayerState& L, uint32_t i, uint32_t lo, uint32_t hi, bool pack, LayerArgs a, cudaStream_t s);
int ssd_join_deferred(kvpool* p, cudaStream_t s);  // end of a batched offload: `s` waits for the pack launches of the SSD-type devices
int ssd_wait_stored(kvpool* p, const LayerState& L, cudaStream_t s);  // `s` waits until the layer's store commands have completed
int ssd_drain(kvpool* p);                                           // host waits for every worker; EIO if a command failed
int ssd_read(kvpool* p, uint32_t i, uint64_t off, void* dst, uint64_t n);  // after ssd_drain
int ssd_measure(kvpool* p, uint32_t i, bool write, uint64_t bytes, uint32_t iters, double* gbps);
inline bool all_hbm(const kvpool* p) { return p->hbm_mask == (p->n >= 32 ? 0xFFFFFFFFu : (1u << p->n) - 1u); }

}  // namespace kvp
