// KV-passthrough, host side: one SSD-type pool device = a block device (or a file standing in for one)
// opened O_DIRECT and addressed by LBA, a queue of asynchronous store / retrieve commands, and the device's own worker
// thread ("each pool device has its own worker thread") that polls for the GPU's half of each command and
// completes it — submission (the API call) is decoupled from completion (the worker).  The worker drives the disk through
// an io_uring of its own (raw system calls, no liburing): it submits the read / write of every command whose GPU half has
// arrived and reaps completions from the ring, so that several commands of one device are in flight at once (as many as
// it has lanes) while commands that touch the same sectors keep their order; where the kernel has no io_uring (or with
// KVPOOL_SSD_SYNC=1 in the environment) it falls back to one synchronous pread / pwrite at a time.
// Pure C++17, no CUDA: the bounce memory and the GPU<->CPU sequence flags are handed in by kvpool_ssd.cu.
#pragma once
#include <atomic>
#include <condition_variable>
#include <cstdint>
#include <deque>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

namespace kvp {

// ceil(set_size * kv_size / sector) sectors; false on a zero sector size or a result that overflows.
bool lba_range_len(uint64_t set_size, uint64_t kv_size, uint64_t sector, uint64_t* n_sectors);

// Wrap-aware "flag has reached v" on a 32-bit sequence number (the comparison cuStreamWaitValue32 GEQ makes).
inline bool seq_reached(const volatile uint32_t* f, uint32_t v) {
  return static_cast<int32_t>(__atomic_load_n(f, __ATOMIC_ACQUIRE) - v) >= 0;
}

struct SsdCmd {
  enum Op : uint8_t { kRead, kWrite };
  Op op;
  bool zero_tail;     // write: the command ends its LBA range — what is left of the last sector is zero (R18)
  uint32_t lane, use; // bounce lane of that direction and the lane's use number (1, 2, ...)
  uint64_t file_off;  // byte offset of the first sector touched (a multiple of the sector size)
  uint32_t head;      // the payload starts `head` bytes into that sector (0 whenever KV_size is a multiple of the sector)
  uint64_t len;       // payload bytes, at bounce + head
};

// The kernel's asynchronous I/O rings, set up and driven with raw system calls (io_uring_setup / io_uring_enter + mmap).
class Uring {
 public:
  ~Uring() { close(); }
  bool open(unsigned entries);  // false: io_uring is not available here
  void close();
  bool ok() const { return fd_ >= 0; }
  // queue one read / write of `len` bytes (false: the submission ring is full); flush() hands queued entries to the kernel
  bool queue(bool write, int file, void* buf, uint32_t len, uint64_t off, uint64_t user_data);
  int flush();
  unsigned drop_unsubmitted();  // after a failed flush(): take the entries the kernel did not accept off the ring; how many
  bool reap(uint64_t* user_data, int32_t* res);  // one completion, if any
  int wait_one();                                // sleep in the kernel until a completion is there
 private:
  int fd_ = -1;
  unsigned entries_ = 0, to_submit_ = 0;
  void *sq_ring_ = nullptr, *cq_ring_ = nullptr, *sqes_ = nullptr;
  size_t sq_ring_bytes_ = 0, cq_ring_bytes_ = 0, sqes_bytes_ = 0;
  unsigned *sq_head_ = nullptr, *sq_tail_ = nullptr, *sq_mask_ = nullptr, *sq_array_ = nullptr;
  unsigned *cq_head_ = nullptr, *cq_tail_ = nullptr, *cq_mask_ = nullptr;
  void* cqes_ = nullptr;
};

class SsdDevice {
 public:
  ~SsdDevice() { close(); }
  // Opens `path` O_DIRECT (a block device: capacity must fit it; a regular file: created / grown to `capacity`).
  // sector 0 = ask the block device (BLKSSZGET), 4096 for a file.  Falls back to buffered I/O where the file system
  // refuses O_DIRECT (direct() says which).  Returns 0 or a negative KVPOOL_E* code with *err set.
  int open(const char* path, uint64_t capacity, uint32_t sector, std::string* err);
  void close();
  // The bounce lanes of both directions (0 = retrieve, 1 = offload): lane k of direction d is lane_bytes of pinned
  // memory at bounce[d] + k*lane_bytes; gpu_seq[d][k*stride] is written by the GPU stream, cpu_seq[d][k*stride] by the
  // worker (32-bit sequence numbers, `stride` words apart).  Starts the worker.
  void start(uint32_t n_lanes, uint64_t lane_bytes, uint8_t* const bounce[2], volatile uint32_t* const gpu_seq[2],
             volatile uint32_t* const cpu_seq[2], uint32_t stride);
  void stop();  // drains, then joins the worker
  void submit(const SsdCmd& c);
  void drain();  // block until every submitted command has completed
  void abort() { abort_.store(true); }  // the GPU is gone: commands still waiting for its half fail with ECANCELED instead of polling on
  // first I/O error since the last call (an errno value; 0 = none).  A failed command still completes its handshake,
  // so that no stream waits for ever.
  int take_error() { return error_.exchange(0); }
  // commands that have failed since start (never reset; readable at any time from any thread)
  uint64_t failed() const { return failed_.load(); }
  // Synchronous helpers for inspection / measurement (call after drain()): whole sectors are moved through `scratch`
  // (4 KiB-aligned, scratch_bytes a multiple of the sector size).
  int read_bytes(uint64_t off, void* dst, uint64_t n, uint8_t* scratch, uint64_t scratch_bytes);
  int io_span(bool write, uint64_t off, uint64_t n, uint8_t* scratch, uint64_t scratch_bytes);  // n bytes in scratch-sized commands
  uint32_t sector() const { return sector_; }
  uint64_t capacity() const { return capacity_; }
  bool direct() const { return direct_; }
  bool block_device() const { return blockdev_; }
  uint64_t completed(int write) const { return done_[write ? 1 : 0].load(); }
  bool running() const { return worker_.joinable(); }
  unsigned queue_depth() const { return depth_; }  // commands the worker keeps in flight (1 = the synchronous fall-back)

 private:
  void run();
  void run_async();
  struct Active;  // a command the asynchronous worker has taken off the queue
  bool gpu_half_arrived(const SsdCmd& c) const;
  int prepare_store(const SsdCmd& c);  // first / last sector of a store: keep the neighbours' bytes, or zero the padding
  void complete(const SsdCmd& c, int err, bool lane_is_ours);  // lane_is_ours: the GPU's half of the command had arrived
  bool wait_flag(const volatile uint32_t* f, uint32_t v);
  int rw_full(bool write, uint64_t off, uint8_t* buf, uint64_t n);
  void execute(const SsdCmd& c);

  int fd_ = -1;
  uint32_t sector_ = 0;
  uint64_t capacity_ = 0;
  bool direct_ = false, blockdev_ = false, created_ = false;
  std::string path_;
  uint32_t n_lanes_ = 0, stride_ = 0;
  uint64_t lane_bytes_ = 0;
  uint8_t* bounce_[2] = {nullptr, nullptr};
  volatile uint32_t* gpu_seq_[2] = {nullptr, nullptr};
  volatile uint32_t* cpu_seq_[2] = {nullptr, nullptr};
  uint8_t* edge_ = nullptr;  // one aligned sector for read-modify-write of a command's first / last sector
  std::thread worker_;
  std::mutex mu_;
  std::condition_variable cv_, cv_done_;
  std::deque<SsdCmd> q_;
  uint64_t submitted_ = 0, finished_ = 0;
  bool stopping_ = false;
  std::atomic<int> error_{0};
  std::atomic<uint64_t> failed_{0};
  std::atomic<bool> abort_{false};
  Uring ring_;
  unsigned depth_ = 1;
  std::atomic<uint64_t> done_[2] = {{0}, {0}};
};

}  // namespace kvp
