// libkvpool.so: SSD-type pool devices — KV-passthrough, GPU side.  DESIGN.md section 13.
//
// An SSD-type device's share of a layer moves in lane-sized commands, DEVICE-MAJOR (runs of consecutive slots of its
// stripe = consecutive bytes of its LBA range, reached through the device's inverse map like the chunks of kvpool_xfer.cu):
//
//   store    (Alg. 1 l.20-21, SSD_Direct_Store):    pack kernel -> lane.bounce (mapped pinned memory, written over the link)
//                                                    -> the device's worker writes the LBA range (ssd_io.cpp)
//   retrieve (SSD_Direct_Retrieve):   worker reads the LBA range -> lane.bounce -> unpack kernel (reads it
//                                                    over the link)
//
// The GPU streams and the worker never synchronise with the host: each lane and direction has two 32-bit sequence flags in
// mapped pinned memory — gpu_seq, raised by a stream write-value behind the lane's kernel, and cpu_seq, raised by the worker
// behind its read / write — and each side waits for the other with a stream wait-value / a poll.  The API call only
// enqueues: stream operations on the GPU side, one command on the worker's queue.
//
// No copy engine on this path, on purpose.  A first version staged every lane through an HBM piece and a cudaMemcpyAsync
// (pack -> HBM -> D2H -> bounce), with the wait-value in front of the copy.  A wait-value that precedes a copy sits on the
// copy engine's channel, and while it waits for the disk it holds up the copies of OTHER streams on that engine: next to a
// host-memory device's 200 MiB copies the lanes' 8 MiB copies fell from 5 to 0.2-2.9 GB/s (an offload of host + SSD moved
// 25-45 GB/s instead of 54), and two pools on two host threads stopped making progress altogether.  On a compute stream a
// waiting wait-value holds up nothing but its own stream.  The disk is ten times slower than SM-issued transfers over the
// link (51 GB/s), so the kernels lose nothing by reaching the bounce memory themselves.
#include "kvpool_internal.hpp"

namespace kvp {
namespace {

// cuStreamWaitValue32 / cuStreamWriteValue32 (driver API), reached through the runtime's entry-point query so that the
// library links against cudart only.  CUstream = cudaStream_t, CUdeviceptr = unsigned long long, CUresult 0 = success.
using MemOpFn = int (*)(cudaStream_t, unsigned long long, unsigned int, unsigned int);
MemOpFn g_wait_value = nullptr, g_write_value = nullptr;
constexpr unsigned int kWaitGeq = 0x0, kWriteDefault = 0x0;  // CU_STREAM_WAIT_VALUE_GEQ (wrap-aware), CU_STREAM_WRITE_VALUE_DEFAULT (fenced)

}  // namespace

int stream_wait_geq(cudaStream_t s, uint64_t dev_addr, uint32_t value) {
  return g_wait_value(s, dev_addr, value, kWaitGeq) == 0 ? KVPOOL_OK : fail(KVPOOL_ECUDA, "cuStreamWaitValue32 failed");
}
int stream_write(cudaStream_t s, uint64_t dev_addr, uint32_t value) {
  return g_write_value(s, dev_addr, value, kWriteDefault) == 0 ? KVPOOL_OK : fail(KVPOOL_ECUDA, "cuStreamWriteValue32 failed");
}

int memops_init() {
  if (g_wait_value && g_write_value) return KVPOOL_OK;
  void *w = nullptr, *r = nullptr;
  cudaDriverEntryPointQueryResult qw, qr;
  CU(cudaGetDriverEntryPointByVersion("cuStreamWaitValue32", &w, 12000, cudaEnableDefault, &qw));
  CU(cudaGetDriverEntryPointByVersion("cuStreamWriteValue32", &r, 12000, cudaEnableDefault, &qr));
  if (!w || !r || qw != cudaDriverEntryPointSuccess || qr != cudaDriverEntryPointSuccess)
    return fail(KVPOOL_ECUDA, "this driver has no stream memory operations (cuStreamWaitValue32 / cuStreamWriteValue32)");
  g_wait_value = reinterpret_cast<MemOpFn>(w);
  g_write_value = reinterpret_cast<MemOpFn>(r);
  return KVPOOL_OK;
}

namespace {

#define DRV(call)                                                                         \
  do {                                                                                    \
    const int r__ = (call);                                                               \
    if (r__ != 0) return fail(KVPOOL_ECUDA, "%s: driver error %d", #call, r__);           \
  } while (0)

// Flags of lane k, direction d: 32 words per lane (gpu_seq at word 0, cpu_seq at word 16: separate cache lines).
constexpr uint32_t kFlagStride = 32;
inline uint32_t flag_word(const SsdState& S, int d, uint32_t lane, bool cpu) { return (static_cast<uint32_t>(d) * S.n_lanes + lane) * kFlagStride + (cpu ? 16u : 0u); }
inline unsigned long long flag_dev(const SsdState& S, int d, uint32_t lane, bool cpu) { return S.flags_dev + 4ull * flag_word(S, d, lane, cpu); }

void free_lanes(SsdState& S) {
  S.io.stop();
  for (auto& v : S.lane) v.clear();
  for (int d = 0; d < 2; ++d) {
    if (S.kstream[d]) cudaStreamDestroy(S.kstream[d]);
    if (S.fork[d]) cudaEventDestroy(S.fork[d]);
    if (S.join[d]) cudaEventDestroy(S.join[d]);
    S.kstream[d] = nullptr;
    S.fork[d] = S.join[d] = nullptr;
  }
  if (S.bounce_base) cudaFreeHost(S.bounce_base);
  if (S.flags) cudaFreeHost(S.flags);
  S.bounce_base = nullptr;
  S.flags = nullptr;
  S.n_lanes = 0;
}

uint64_t gcd64(uint64_t a, uint64_t b) {
  while (b) { const uint64_t t = a % b; a = b; b = t; }
  return a;
}

}  // namespace

int ssd_open(kvpool* p, uint32_t i, const kvpool_device_desc& d) {
  int rc = memops_init();
  if (rc != KVPOOL_OK) return rc;
  std::unique_ptr<SsdState> S(new SsdState);
  std::string err;
  rc = S->io.open(d.path, d.capacity_bytes, d.sector_bytes, &err);
  if (rc != KVPOOL_OK) return fail(rc, "create: pool device %u: %s", i, err.c_str());
  S->scratch = static_cast<uint8_t*>(aligned_alloc(4096, kSsdScratchBytes));
  if (!S->scratch) return fail(KVPOOL_ENOMEM, "create: pool device %u: out of memory", i);
  p->ssd[i] = std::move(S);
  p->ssd_mask |= 1u << i;
  return KVPOOL_OK;
}

void ssd_close_all(kvpool* p) {
  for (auto& S : p->ssd) {
    if (!S) continue;
    free_lanes(*S);
    S->io.close();
    free(S->scratch);
    S.reset();
  }
  p->ssd_mask = 0;
}

int ssd_ensure_lanes(kvpool* p) {
  for (uint32_t i = 0; i < p->n; ++i) {
    if (!is_ssd(p, i)) continue;
    SsdState& S = *p->ssd[i];
    if (S.n_lanes) continue;
    const uint64_t sec = S.io.sector();
    // a command carries at least one KV cache, displaced by up to a sector and rounded up to one
    const uint64_t least = (p->payload + sec - 1) / sec * sec + 2 * sec;
    S.lane_bytes = (std::max<uint64_t>(p->tune.ssd_chunk_bytes, least) + 4095) / 4096 * 4096;
    const uint32_t n = std::max<uint32_t>(p->tune.ssd_lanes, 1);
    const uint64_t total = 2ull * n * S.lane_bytes;
    cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&S.bounce_base), total, cudaHostAllocPortable | cudaHostAllocMapped);
    void* bd = nullptr;
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&bd, S.bounce_base, 0);
    if (e == cudaSuccess) e = cudaHostAlloc(reinterpret_cast<void**>(&S.flags), 2ull * n * kFlagStride * 4, cudaHostAllocMapped | cudaHostAllocPortable);
    void* fd = nullptr;
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&fd, S.flags, 0);
    if (e != cudaSuccess) {
      cudaGetLastError();
      free_lanes(S);
      return fail(KVPOOL_ENOMEM, "place: bounce lanes of SSD-type device %u (%llu bytes pinned): %s", i, (unsigned long long)total, cudaGetErrorString(e));
    }
    memset(S.flags, 0, 2ull * n * kFlagStride * 4);
    S.flags_dev = reinterpret_cast<uint64_t>(fd);
    S.n_lanes = n;  // (flag_word needs it) every failure below goes through free_lanes, which takes it back to 0:
                    // n_lanes != 0 on return means lanes, streams and a running worker
    for (int d = 0; d < 2 && e == cudaSuccess; ++d) {
      e = cudaStreamCreateWithFlags(&S.kstream[d], cudaStreamNonBlocking);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&S.fork[d], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&S.join[d], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {  // nothing half-made is left behind: the next kvpool_place starts over
      cudaGetLastError();
      free_lanes(S);
      return fail(KVPOOL_ECUDA, "place: streams / events of SSD-type device %u: %s", i, cudaGetErrorString(e));
    }
    for (int d = 0; d < 2; ++d) {
      S.lane[d].resize(n);
      for (uint32_t k = 0; k < n; ++k) {
        SsdLane& ln = S.lane[d][k];
        ln.bounce = S.bounce_base + (static_cast<uint64_t>(d) * n + k) * S.lane_bytes;
        ln.bounce_dev = static_cast<uint8_t*>(bd) + (static_cast<uint64_t>(d) * n + k) * S.lane_bytes;
      }
    }
    uint8_t* const bounce[2] = {S.lane[0][0].bounce, S.lane[1][0].bounce};
    volatile uint32_t* const gpu[2] = {S.flags + flag_word(S, 0, 0, false), S.flags + flag_word(S, 1, 0, false)};
    volatile uint32_t* const cpu[2] = {S.flags + flag_word(S, 0, 0, true), S.flags + flag_word(S, 1, 0, true)};
    S.io.start(n, S.lane_bytes, bounce, gpu, cpu, kFlagStride);
  }
  return KVPOOL_OK;
}

namespace {

// One command of device i: `bytes` at byte offset `byte0` of the device travel between its LBA range and the bounce memory of
// the next lane of that direction.  `launch(at)` enqueues on `s` the launch that fills (store) or drains (retrieve) the lane
// at its GPU address `at` and returns a KVPOOL code.  *lane_out / *use_out name the command (for ssd_wait_stored).
template <class Launch>
int ssd_command(kvpool* p, uint32_t i, bool pack, uint64_t byte0, uint64_t bytes, bool zero_tail, cudaStream_t s, Launch&& launch,
                uint32_t* lane_out, uint32_t* use_out) {
  SsdState& S = *p->ssd[i];
  const uint64_t sec = S.io.sector();
  const int d = pack ? 1 : 0;
  const uint64_t at = byte0 / sec * sec;
  const uint32_t head = static_cast<uint32_t>(byte0 - at);
  const uint32_t k = S.cursor[d]++ % S.n_lanes;
  SsdLane& ln = S.lane[d][k];
  const uint32_t u = ++ln.uses;
  *lane_out = k;
  *use_out = u;
  // If enqueueing fails half way, both flags of this use are raised from the host so that no later use of the lane (and no
  // worker) waits for a hand-over that will never come.  Earlier uses of the lane may still be pending, and their own
  // hand-overs (a stream write-value of u-1, the worker's store of u-1) land later: a plain store here could be overwritten
  // by them and the flag would read u-1 for ever.  So the host first waits until both flags have reached u-1 — the earlier
  // uses are enqueued and complete by themselves — and only then raises them to u; flags never go backwards.  (If the GPU
  // itself is gone the wait gives up after two seconds and the pool's abort path takes over at kvpool_destroy.)
  auto abandon = [&](int rc) {
    for (int cpu = 0; cpu < 2; ++cpu) {
      volatile uint32_t* f = S.flags + flag_word(S, d, k, cpu != 0);
      const timespec nap{0, 50000};
      for (int spins = 0; spins < 40000 && !seq_reached(f, u - 1); ++spins) nanosleep(&nap, nullptr);
      __atomic_store_n(f, u, __ATOMIC_RELEASE);
    }
    return rc;
  };
  int rc;
  // The kernel itself moves the bytes between the paged blocks and the lane's mapped bounce memory over the link; the two
  // hand-overs are stream memory operations on the kernel's own stream.
  uint8_t* const at_dev = ln.bounce_dev + head;
  if (pack) {
    // SSD_Direct_Store: once the lane's previous command is on the disk (cpu_seq >= u-1) gather into the bounce memory,
    // then tell the worker (gpu_seq = u, fenced: the kernel's stores are visible to the CPU first)
    if (g_wait_value(s, flag_dev(S, d, k, true), u - 1, kWaitGeq) != 0) return abandon(fail(KVPOOL_ECUDA, "cuStreamWaitValue32 failed"));
    if ((rc = launch(at_dev)) != KVPOOL_OK) return abandon(rc);
    if (g_write_value(s, flag_dev(S, d, k, false), u, kWriteDefault) != 0) return abandon(fail(KVPOOL_ECUDA, "cuStreamWriteValue32 failed"));
    S.io.submit(SsdCmd{SsdCmd::kWrite, zero_tail, k, u, at, head, bytes});
    return KVPOOL_OK;
  }
  // SSD_Direct_Retrieve: the worker reads the LBA range into the bounce memory once the lane's previous command has been
  // scattered (gpu_seq >= u-1) and raises cpu_seq = u; the unpack waits for that and frees the lane (gpu_seq = u)
  S.io.submit(SsdCmd{SsdCmd::kRead, false, k, u, at, head, bytes});
  if (g_wait_value(s, flag_dev(S, d, k, true), u, kWaitGeq) != 0) return abandon(fail(KVPOOL_ECUDA, "cuStreamWaitValue32 failed"));
  if ((rc = launch(at_dev)) != KVPOOL_OK) return abandon(rc);
  if (g_write_value(s, flag_dev(S, d, k, false), u, kWriteDefault) != 0) return abandon(fail(KVPOOL_ECUDA, "cuStreamWriteValue32 failed"));
  return KVPOOL_OK;
}

}  // namespace

int ssd_move(kvpool* p, LayerState& L, uint32_t i, uint32_t lo, uint32_t hi, bool pack, LayerArgs a, cudaStream_t s) {
  SsdState& S = *p->ssd[i];
  if (!S.n_lanes) return fail(KVPOOL_ESTATE, "SSD-type device %u has no bounce lanes", i);
  const uint64_t P = p->payload, sec = S.io.sector();
  const uint64_t unit = sec / gcd64(P, sec);  // every `unit` KV caches the stripe is back on a sector boundary
  a.order = L.map->order_d;
  a.visit = nullptr;
  // The launches go to the device's own kernel stream, which first catches up with the caller's stream (the source blocks /
  // the destination tensor are whatever `s` has made of them so far) and is joined back below.  On `s` itself they would
  // sit, waiting for lanes the disk frees at its own pace, in front of the next launches of the host-memory devices.
  const int d = pack ? 1 : 0;
  cudaStream_t k = S.kstream[d];
  CU(cudaEventRecord(S.fork[d], s));
  CU(cudaStreamWaitEvent(k, S.fork[d], 0));
  for (uint32_t x = lo; x < hi;) {
    const uint64_t byte0 = L.stripe_off[i] + static_cast<uint64_t>(x) * P;
    const uint32_t head = static_cast<uint32_t>(byte0 % sec);
    uint32_t n = static_cast<uint32_t>(std::min<uint64_t>(hi - x, (S.lane_bytes - sec - head) / P));
    if (unit > 1 && x + n < hi) {  // ragged KV size: end the command on a sector boundary when one is within reach
      const uint64_t end = (static_cast<uint64_t>(x) + n) / unit * unit;
      if (end > x) n = static_cast<uint32_t>(end - x);
    }
    a.j0 = L.map->start[i] + x;
    a.K = n;
    uint32_t lane = 0, use = 0;
    const int rc = ssd_command(p, i, pack, byte0, static_cast<uint64_t>(n) * P, x + n == L.map->counts[i], k,
                               [&](uint8_t* at) {
                                 a.pool_base[0] = reinterpret_cast<uint64_t>(at);
                                 return launch_counted(p, a, pack, true, k, true);  // a link-bound launch: 4 CTAs fill the link
                               },
                               &lane, &use);
    if (rc != KVPOOL_OK) {  // what has been launched so far still reads / writes the caller's blocks: join it before giving up
      if (cudaEventRecord(S.join[d], k) == cudaSuccess) cudaStreamWaitEvent(s, S.join[d], 0);
      cudaGetLastError();
      return rc;
    }
    if (pack) {
      auto& uses = L.ssd_lane_use[i];
      if (uses.size() < S.n_lanes) uses.resize(S.n_lanes, 0);
      uses[lane] = use;  // uses of a lane only grow
      L.ssd_stored |= 1u << i;
    }
    x += n;
  }
  // join: a retrieve is complete in `s` order (kvpool.h), and work enqueued on `s` after an offload may overwrite the source
  // blocks - per layer for the per-layer calls, once at the end of a batched offload (the source blocks of all its layers
  // stay as they are until the call's last launch anyway)
  CU(cudaEventRecord(S.join[d], k));
  if (pack && p->ssd_defer_join) S.join_pending = true;
  else CU(cudaStreamWaitEvent(s, S.join[d], 0));
  return KVPOOL_OK;
}

int ssd_join_deferred(kvpool* p, cudaStream_t s) {
  for (auto& S : p->ssd) {
    if (!S || !S->join_pending) continue;
    S->join_pending = false;
    CU(cudaStreamWaitEvent(s, S->join[1], 0));
  }
  return KVPOOL_OK;
}

int ssd_wait_stored(kvpool* p, const LayerState& L, cudaStream_t s) {
  for (uint32_t i = 0; i < p->n; ++i) {
    if (!(L.ssd_stored >> i & 1u)) continue;
    const SsdState& S = *p->ssd[i];
    const auto& uses = L.ssd_lane_use[i];
    for (uint32_t k = 0; k < uses.size(); ++k) {  // every lane that carried a piece of the stripe, not just the last one
      if (uses[k] == 0 || seq_reached(S.flags + flag_word(S, 1, k, true), uses[k])) continue;  // none, or already on the disk
      DRV(g_wait_value(s, flag_dev(S, 1, k, true), uses[k], kWaitGeq));
    }
  }
  return KVPOOL_OK;
}

int ssd_drain(kvpool* p) {
  int err = 0;
  for (auto& S : p->ssd) {
    if (!S) continue;
    if (S->io.running()) S->io.drain();
    const int e = S->io.take_error();
    if (e && !err) err = e;
  }
  return err ? fail(KVPOOL_EIO, "an SSD-type pool device failed a store / retrieve command: %s", strerror(err)) : KVPOOL_OK;
}

int ssd_read(kvpool* p, uint32_t i, uint64_t off, void* dst, uint64_t n) {
  SsdState& S = *p->ssd[i];
  const int e = S.io.read_bytes(off, dst, n, S.scratch, kSsdScratchBytes);
  return e ? fail(KVPOOL_EIO, "read of SSD-type device %u: %s", i, strerror(e)) : KVPOOL_OK;
}

// "Measured bandwidth" of an SSD-type device, with the mechanism that moves the bytes: the first `bytes` of
// the device travel through the device's own lanes — worker, bounce memory, link, gather / scatter kernel — exactly as a
// retrieve (or an offload) moves them, between the disk and a scratch paged layout whose block table and inverse map are
// the identity; median of `iters` passes by the host's clock around enqueue + completion.  (A plain pread loop into a
// cache-resident buffer reads 10-15 % fast.)  The region is written once first, so that a sparse stand-in file has its blocks.
int ssd_measure(kvpool* p, uint32_t i, bool write, uint64_t bytes, uint32_t iters, double* gbps) {
  int rc = ssd_ensure_lanes(p);
  if (rc != KVPOOL_OK) return rc;
  SsdState& S = *p->ssd[i];
  DeviceGuard guard(p->cuda_device);
  const uint64_t P = p->payload, sec = S.io.sector();
  const uint64_t unit = sec / gcd64(P, sec);                             // KV caches per sector-aligned run
  const uint64_t K = (S.lane_bytes - 2 * sec) / (unit * P) * unit;       // KV caches per command: a whole number of sectors
  if (K == 0 || K > 0x7fffffffull) return fail(KVPOOL_EINVAL, "measure_bandwidth: the lanes of SSD-type device %u are too small for a sector-aligned run of KV caches", i);
  const uint64_t piece = K * P;
  bytes = bytes / piece * piece;
  if (bytes == 0) return fail(KVPOOL_EINVAL, "measure_bandwidth: fewer bytes than one command (%llu)", (unsigned long long)piece);
  struct Scratch {
    void* buf = nullptr;
    uint32_t* ident = nullptr;
    ~Scratch() {
      if (buf) cudaFree(buf);
      if (ident) cudaFree(ident);
    }
  } m;
  CU(cudaMalloc(&m.buf, piece));
  CU(cudaMalloc(reinterpret_cast<void**>(&m.ident), K * 4));
  std::vector<uint32_t> h(K);
  std::iota(h.begin(), h.end(), 0u);
  cudaStream_t s = p->upload;
  CU(cudaMemcpyAsync(m.ident, h.data(), K * 4, cudaMemcpyHostToDevice, s));
  CU(cudaMemsetAsync(m.buf, 0x5a, piece, s));
  CU(cudaStreamSynchronize(s));
  LayerArgs a{};
  a.k_base = static_cast<uint8_t*>(m.buf);
  a.v_base = static_cast<uint8_t*>(m.buf) + K * p->kvb;
  a.stride = p->kvb;
  a.table = reinterpret_cast<const int32_t*>(m.ident);
  a.order = m.ident;
  a.K = static_cast<uint32_t>(K);
  a.kvb = static_cast<uint32_t>(p->kvb);
  std::vector<double> sec_s(iters);
  for (uint32_t it = 0; it < iters + 1; ++it) {  // pass 0 writes the region (and warms up)
    const bool w = write || it == 0;
    timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    for (uint64_t off = 0; off < bytes; off += piece) {
      uint32_t lane, use;
      rc = ssd_command(p, i, w, off, piece, false, s,
                       [&](uint8_t* at) {
                         a.pool_base[0] = reinterpret_cast<uint64_t>(at);
                         return launch_counted(p, a, w, true, s, true);
                       },
                       &lane, &use);
      if (rc != KVPOOL_OK) return rc;
    }
    CU(cudaStreamSynchronize(s));
    if ((rc = ssd_drain(p)) != KVPOOL_OK) return rc;
    clock_gettime(CLOCK_MONOTONIC, &t1);
    if (it > 0) sec_s[it - 1] = (t1.tv_sec - t0.tv_sec) + 1e-9 * (t1.tv_nsec - t0.tv_nsec);
  }
  std::sort(sec_s.begin(), sec_s.end());
  *gbps = static_cast<double>(bytes) / (sec_s[iters / 2] * 1.0e9);
  return KVPOOL_OK;
}

}  // namespace kvp
