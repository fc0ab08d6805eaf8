// libkvpool.so, part 1 of 3 (include/kvpool.h): pool life cycle, bandwidth measurement, placement + GLT (a1-a4), introspection,
// and the helpers every part shares (kvpool_internal.hpp).  The hot path is kvpool_xfer.cu, the development entry points
// of include/kvpool_dev.h are kvpool_dev.cu, device code lives in kernels.cu.
#include "kvpool_internal.hpp"

using namespace kvp;

namespace kvp {

namespace {
thread_local std::string g_err;
}

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

const char* last_error_message() { return g_err.c_str(); }

PoolLock::PoolLock(kvpool* p) {
  if (p) l = std::unique_lock<std::recursive_mutex>(p->mu);
}

void default_tuning(kvpool* p) {
  p->tune.kernel = KVPOOL_KERNEL_VEC16;
  p->tune.link_kernel = KVPOOL_KERNEL_BULK;  // 2 CTAs already saturate the link (profiles/r1_sweep_link.txt)
  p->tune.hbm_ctas = 16u * p->sm_count;  // many short CTAs balance the tail better than a persistent grid here (profiles/r1_sweep_hbm.txt)
  p->tune.link_ctas = 4;
  p->tune.bulk_chunk = 16384;  // 3 issuing lanes per SM x 4 stages x 16 KiB = 192 KiB of shared memory, 144 KiB of loads in flight per SM:
  p->tune.bulk_stages = 4;     // 6.2 / 6.3 TB/s pack / unpack in-device; 2 lanes x 6 stages (more bytes in flight, fewer issue slots)
  p->tune.bulk_warps = 3;      // reads 5.9 / 5.8 (profiles/r3_sweep_bulk.txt)
  p->tune.stage_slots = 2;                   // one slot fills while the other drains; the kernels take ~2 % of a copy's time
  p->tune.stage_chunk_bytes = 256ull << 20;  // ring <= 512 MiB whatever the context length (larger layers: device-major chunks)
  p->tune.vec_threads = 512;
  p->tune.vec_unroll = 8;
  p->tune.group_bytes = 64ull << 20;
  p->tune.auto_threshold_bytes = 8ull << 20;
  p->tune.pdl = 1;
  p->tune.ssd_lanes = 4;
  p->tune.ssd_chunk_bytes = 8ull << 20;
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


LaunchCfg launch_cfg(const kvpool* p, bool link_bound, bool pack, bool lane) {
  // a zero-copy launch over a pool with HBM devices moves most of its bytes at HBM / NVLink rates: give it the HBM grid
  // (not a launch on an SSD-type device's lane: that one touches nothing but the lane's mapped host memory)
  if (p->hbm_mask && !lane) link_bound = false;
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


// Does a transfer of `host_bytes` to / from host-memory devices go through the staging ring and the copy engines?
bool use_staged(const kvpool* p, bool pack, uint64_t host_bytes) {
  if (p->ssd_mask) return true;   // a pool with an SSD-type device moves device-major on every path (kvpool_ssd.cu)
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

}  // namespace kvp

extern "C" {

const char* kvpool_last_error(void) { return last_error_message(); }
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
    if (devs[i].flags & ~(KVPOOL_DEV_WRITE_COMBINED | KVPOOL_DEV_NUMA_STRICT | KVPOOL_DEV_HBM | KVPOOL_DEV_CUDA_HOSTALLOC | KVPOOL_DEV_SSD)) return fail(KVPOOL_EINVAL, "create: device %u unknown flags", i);
    if ((devs[i].flags & KVPOOL_DEV_HBM) && (devs[i].flags & ~KVPOOL_DEV_HBM)) return fail(KVPOOL_EINVAL, "create: device %u: KVPOOL_DEV_HBM excludes the host-memory flags", i);
    if ((devs[i].flags & KVPOOL_DEV_SSD) && (devs[i].flags & ~KVPOOL_DEV_SSD)) return fail(KVPOOL_EINVAL, "create: device %u: KVPOOL_DEV_SSD excludes every other flag", i);
    if ((devs[i].flags & KVPOOL_DEV_SSD) && (!devs[i].path || !*devs[i].path)) return fail(KVPOOL_EINVAL, "create: device %u: an SSD-type device needs a path", i);
    if (!(devs[i].flags & KVPOOL_DEV_SSD) && (devs[i].path || devs[i].sector_bytes)) return fail(KVPOOL_EINVAL, "create: device %u: path / sector_bytes are for SSD-type devices", i);
    if (devs[i].reserved) return fail(KVPOOL_EINVAL, "create: device %u: reserved must be 0", i);
    for (uint32_t j = 0; j < i && (devs[i].flags & KVPOOL_DEV_SSD); ++j)
      if ((devs[j].flags & KVPOOL_DEV_SSD) && strcmp(devs[j].path, devs[i].path) == 0)
        return fail(KVPOOL_EINVAL, "create: devices %u and %u name the same path: their LBA ranges would overlap", j, i);
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
    ssd_close_all(p.get());
    for (auto& b : p->bufs) host_buffer_free(&b);
    for (auto s : p->own_streams) cudaStreamDestroy(s);
    if (p->table_arena) cudaFree(p->table_arena);
    if (p->table_arena_host) cudaFreeHost(p->table_arena_host);
    if (p->upload) cudaStreamDestroy(p->upload);
    if (p->join_out) cudaStreamDestroy(p->join_out);
  };
  p->bufs.resize(n_devs);
  p->ssd.resize(n_devs);
  for (uint32_t i = 0; i < n_devs; ++i) {
    std::string err;
    if (devs[i].flags & KVPOOL_DEV_SSD) {  // block storage: no buffer; LBAs are handed out in units of its sector size
      const int rc = ssd_open(p.get(), i, devs[i]);
      if (rc != KVPOOL_OK) { const std::string keep = last_error_message(); cleanup(); return fail(rc, "%s", keep.c_str()); }
      p->bufs[i].bytes = p->ssd[i]->io.capacity();
      p->alloc.emplace_back(p->bufs[i].bytes, std::max<uint64_t>(4096, p->ssd[i]->io.sector()));
      continue;
    }
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
    for (uint32_t j = 0; j < i && devs[i].link_group && !is_ssd(p.get(), i); ++j)  // (an SSD-type device keeps streams of its own)
      if (devs[j].link_group == devs[i].link_group && !is_ssd(p.get(), j)) { first = j; break; }
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
  if (cudaDeviceSynchronize() != cudaSuccess) {  // a dead GPU never delivers its half of the pending SSD commands
    cudaGetLastError();
    for (auto& S : p->ssd)
      if (S) S->io.abort();
  }
  for (auto* pl : p->live) destroy_placement(p, pl);
  p->live.clear();
  ssd_close_all(p);  // (after the device-wide synchronize above: every command has had the GPU's half)
  free_slots(p);
  for (auto s : p->own_streams) cudaStreamDestroy(s);
  for (auto& x : p->sig) {  // (their streams are in own_streams)
    if (x.mem_d) cudaFree(x.mem_d);
    if (x.done) cudaEventDestroy(x.done);
  }
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
  if (is_ssd(p, dev)) return ssd_measure(p, dev, direction == 1 || direction == KVPOOL_MEASURE_KERNEL_OFFLOAD, bytes, iters, gbps_out);
  DeviceGuard guard(p->cuda_device);
  struct Scratch {  // whatever the measurement allocates goes away on every return path
    void* buf = nullptr;
    uint32_t* ident = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ~Scratch() {
      if (e0) cudaEventDestroy(e0);
      if (e1) cudaEventDestroy(e1);
      if (buf) cudaFree(buf);
      if (ident) cudaFree(ident);
    }
  } m;
  CU(cudaMalloc(&m.buf, bytes));
  CU(cudaEventCreate(&m.e0));
  CU(cudaEventCreate(&m.e1));
  std::vector<float> ms(iters);
  const bool by_kernel = direction >= KVPOOL_MEASURE_KERNEL_RETRIEVE, towards_gpu = direction == 0 || direction == KVPOOL_MEASURE_KERNEL_RETRIEVE;
  cudaStream_t s = towards_gpu ? p->io[dev] : p->io_out[dev];
  // kernel modes: K blocks, block u at slot u of the device's buffer and at physical block u of the scratch paged layout
  // (K plane then V plane): one device-major launch whose inverse map and block table are both the identity
  const uint32_t K = static_cast<uint32_t>(std::min<uint64_t>(bytes / p->payload, 0x7fffffffull));
  LayerArgs ka{};
  if (by_kernel) {
    if (K == 0) return fail(KVPOOL_EINVAL, "measure_bandwidth: fewer bytes than one KV cache (%llu)", (unsigned long long)p->payload);
    bytes = static_cast<uint64_t>(K) * p->payload;
    std::vector<uint32_t> h(K);
    std::iota(h.begin(), h.end(), 0u);
    CU(cudaMalloc(reinterpret_cast<void**>(&m.ident), static_cast<uint64_t>(K) * 4));
    CU(cudaMemcpyAsync(m.ident, h.data(), static_cast<uint64_t>(K) * 4, cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));
    ka.k_base = static_cast<uint8_t*>(m.buf);
    ka.v_base = static_cast<uint8_t*>(m.buf) + static_cast<uint64_t>(K) * p->kvb;
    ka.stride = p->kvb;
    ka.table = reinterpret_cast<const int32_t*>(m.ident);
    ka.order = m.ident;
    ka.K = K;
    ka.kvb = static_cast<uint32_t>(p->kvb);
    ka.pool_base[0] = reinterpret_cast<uint64_t>(p->bufs[dev].dev_alias);
  }
  if (towards_gpu && !is_hbm(p, dev)) {
    // Pages the CPU has just zeroed sit partly in its caches; host->GPU DMA reads of such lines run 5 % slow until a DMA
    // write has claimed them (measured: 52 -> 55.6 GB/s after one pass).  Stripes are always written by an offload
    // before a retrieve reads them, so that is the state to measure: write the region once (no placement is live).
    CU(cudaMemcpyAsync(pool_bytes(p, dev), m.buf, bytes, cudaMemcpyDefault, s));
    p->n_memcpys++;
  }
  for (uint32_t it = 0; it < iters + 1; ++it) {  // first pass is a warm-up
    CU(cudaEventRecord(m.e0, s));
    if (by_kernel) {
      CU(launch_layer_copy(ka, !towards_gpu, launch_cfg(p, !is_hbm(p, dev)), s));
      p->n_kernels++;
    } else {
      CU(towards_gpu ? cudaMemcpyAsync(m.buf, pool_bytes(p, dev), bytes, cudaMemcpyDefault, s)
                     : cudaMemcpyAsync(pool_bytes(p, dev), m.buf, bytes, cudaMemcpyDefault, s));
      p->n_memcpys++;
    }
    CU(cudaEventRecord(m.e1, s));
    CU(cudaStreamSynchronize(s));
    if (it > 0) CU(cudaEventElapsedTime(&ms[it - 1], m.e0, m.e1));
  }
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
  if ((t->ssd_lanes && t->ssd_lanes != d.ssd_lanes) || (t->ssd_chunk_bytes && t->ssd_chunk_bytes != d.ssd_chunk_bytes)) {
    if (t->ssd_lanes > 64) return fail(KVPOOL_EINVAL, "set_tuning: ssd_lanes must be <= 64");
    for (auto& S : p->ssd)
      if (S && S->n_lanes) return fail(KVPOOL_ESTATE, "set_tuning: ssd_lanes / ssd_chunk_bytes are fixed by the first kvpool_place");
    if (t->ssd_lanes) d.ssd_lanes = t->ssd_lanes;
    if (t->ssd_chunk_bytes) d.ssd_chunk_bytes = t->ssd_chunk_bytes;
  }
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
  if (!has_mem(p)) return KVPOOL_OK;  // nothing is ever staged (HBM-type stripes are reached in place, SSD-type devices have lanes)
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
        if (is_mem(p, i)) m->host_blocks += m->counts[i];
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
  // (on an SSD-type device a stripe is an LBA range: it starts on a sector boundary)
  pl->region_off.assign(N, 0);
  pl->region_bytes.assign(N, 0);
  for (uint32_t l = 0; l < L; ++l) {
    auto& Ls = pl->layers[l];
    Ls.stripe_off.assign(N, 0);
    if (p->ssd_mask) Ls.ssd_lane_use.assign(N, {});
    for (uint32_t i = 0; i < N; ++i) {
      const uint64_t align = is_ssd(p, i) ? std::max<uint64_t>(256, p->ssd[i]->io.sector()) : 256;
      Ls.stripe_off[i] = pl->region_bytes[i];  // relative for now
      pl->region_bytes[i] += (static_cast<uint64_t>(Ls.map->counts[i]) * p->payload + align - 1) / align * align;
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
  if (p->ssd_mask) {
    const int rc = ssd_ensure_lanes(p);
    if (rc != KVPOOL_OK) { rollback(); return rc; }
  }
  if ((p->path != KVPOOL_PATH_ZEROCOPY || p->ssd_mask) && has_mem(p)) {
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
  int rc = sync_pool_streams(p);  // the library's own transfers for it must be over
  if (rc != KVPOOL_OK) return rc;
  for (auto& u : pl->last_use) CU(cudaEventSynchronize(u.second));  // and so must the kernels it put on the caller's streams
  rc = p->ssd_mask ? ssd_drain(p) : KVPOOL_OK;  // and the store commands of the SSD-type devices (a failed one: EIO, the placement stays)
  if (rc != KVPOOL_OK) return rc;
  p->live.erase(it);
  destroy_placement(p, pl);
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
  if (type) *type = is_ssd(pl->pool, d) ? KVPOOL_TYPE_SSD : is_hbm(pl->pool, d) ? KVPOOL_TYPE_HBM : KVPOOL_TYPE_MEM;
  if (slot) *slot = s;
  if (host_ptr) {
    if (is_ssd(pl->pool, d))  // Table I: location = LBA (of the sector the payload starts in; kvpool_ssd_location has the byte)
      *host_ptr = reinterpret_cast<void*>(static_cast<uintptr_t>((L.stripe_off[d] + static_cast<uint64_t>(s) * pl->pool->payload) / pl->pool->ssd[d]->io.sector()));
    else *host_ptr = pool_bytes(pl->pool, d) + L.stripe_off[d] + static_cast<uint64_t>(s) * pl->pool->payload;
  }
  return KVPOOL_OK;
}

int kvpool_stripe(const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, void** host_ptr, uint64_t* nbytes) {
  if (!pl || layer >= pl->layers.size() || dev >= pl->pool->n) return fail(KVPOOL_EINVAL, "stripe: bad arguments");
  const LayerState& L = pl->layers[layer];
  const uint64_t bytes = static_cast<uint64_t>(L.map->counts[dev]) * pl->pool->payload;
  if (host_ptr) {
    if (is_ssd(pl->pool, dev)) *host_ptr = reinterpret_cast<void*>(static_cast<uintptr_t>(L.stripe_off[dev] / pl->pool->ssd[dev]->io.sector()));  // first LBA
    else *host_ptr = bytes ? pool_bytes(pl->pool, dev) + L.stripe_off[dev] : nullptr;
  }
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
  if (is_ssd(p, dev)) {  // wait for the device's worker, then read the LBA range with plain preads
    const int rc = ssd_drain(p);
    return rc != KVPOOL_OK ? rc : ssd_read(p, dev, L.stripe_off[dev], dst_host, nbytes);
  }
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
  if (type) *type = is_ssd(p, dev) ? KVPOOL_TYPE_SSD : is_hbm(p, dev) ? KVPOOL_TYPE_HBM : KVPOOL_TYPE_MEM;
  if (gpu) *gpu = p->bufs[dev].gpu;
  return KVPOOL_OK;
}

int kvpool_plan_lba_range(uint64_t set_size, uint64_t kv_size, uint32_t sector_bytes, uint64_t* n_sectors_out) {
  if (!n_sectors_out || !lba_range_len(set_size, kv_size, sector_bytes, n_sectors_out))
    return fail(KVPOOL_EINVAL, "plan_lba_range: null output, zero sector size or a range beyond 2^64 sectors");
  return KVPOOL_OK;
}

int kvpool_ssd_range(const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, uint64_t* first_lba, uint64_t* n_sectors, uint32_t* sector_bytes) {
  if (!pl || layer >= pl->layers.size() || dev >= pl->pool->n) return fail(KVPOOL_EINVAL, "ssd_range: bad arguments");
  if (!is_ssd(pl->pool, dev)) return fail(KVPOOL_EINVAL, "ssd_range: pool device %u is not an SSD-type device", dev);
  const LayerState& L = pl->layers[layer];
  const uint32_t sec = pl->pool->ssd[dev]->io.sector();
  if (first_lba) *first_lba = L.stripe_off[dev] / sec;
  if (n_sectors) lba_range_len(L.map->counts[dev], pl->pool->payload, sec, n_sectors);
  if (sector_bytes) *sector_bytes = sec;
  return KVPOOL_OK;
}

int kvpool_ssd_location(const kvpool_placement_t* pl, uint32_t layer, uint32_t block, uint64_t* lba, uint32_t* byte_in_sector) {
  if (!pl || layer >= pl->layers.size()) return fail(KVPOOL_EINVAL, "ssd_location: bad arguments");
  const LayerState& L = pl->layers[layer];
  if (block >= L.map->K) return fail(KVPOOL_EINVAL, "ssd_location: block %u out of range (K %llu)", block, (unsigned long long)L.map->K);
  const uint32_t d = L.map->dev[block];
  if (!is_ssd(pl->pool, d)) return fail(KVPOOL_EINVAL, "ssd_location: block %u lives on pool device %u, which is not an SSD-type device", block, d);
  const uint64_t sec = pl->pool->ssd[d]->io.sector(), at = L.stripe_off[d] + static_cast<uint64_t>(L.map->slot[block]) * pl->pool->payload;
  if (lba) *lba = at / sec;
  if (byte_in_sector) *byte_in_sector = static_cast<uint32_t>(at % sec);
  return KVPOOL_OK;
}

int kvpool_io_errors(const kvpool_t* p, uint64_t* failed_out) {
  if (!p || !failed_out) return fail(KVPOOL_EINVAL, "io_errors: bad arguments");
  uint64_t n = 0;  // no pool lock: the counters are atomics of the workers, the device list is fixed at create
  for (const auto& S : p->ssd)
    if (S) n += S->io.failed();
  *failed_out = n;
  return KVPOOL_OK;
}

int kvpool_ssd_info(const kvpool_t* p, uint32_t dev, uint32_t* sector_bytes, int32_t* direct_io, int32_t* block_device, uint64_t* stores, uint64_t* retrieves,
                    uint32_t* queue_depth) {
  if (!p || dev >= p->n) return fail(KVPOOL_EINVAL, "ssd_info: bad arguments");
  if (!is_ssd(p, dev)) return fail(KVPOOL_EINVAL, "ssd_info: pool device %u is not an SSD-type device", dev);
  const SsdDevice& io = p->ssd[dev]->io;
  if (sector_bytes) *sector_bytes = io.sector();
  if (direct_io) *direct_io = io.direct();
  if (block_device) *block_device = io.block_device();
  if (stores) *stores = io.completed(1);
  if (retrieves) *retrieves = io.completed(0);
  if (queue_depth) *queue_depth = io.running() ? io.queue_depth() : 0;
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

}  // extern "C"
