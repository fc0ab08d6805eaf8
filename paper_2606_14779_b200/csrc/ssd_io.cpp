// KV-passthrough, host side: see ssd_io.hpp.  SSD_Direct_Store / SSD_Direct_Retrieve of PAPER.md:181-185 with the kernel's
// O_DIRECT block path standing where the paper uses SPDK (no NVMe device and no SPDK in this image: DESIGN.md R19).
#include "ssd_io.hpp"

#include <errno.h>
#include <fcntl.h>
#include <linux/fs.h>
#include <linux/io_uring.h>
#include <sys/ioctl.h>
#include <sys/mman.h>
#include <sys/syscall.h>
#include <sys/stat.h>
#include <time.h>
#include <unistd.h>

#include <algorithm>
#include <chrono>
#include <cstdlib>
#include <cstring>

#include "../../include/kvpool.h"

namespace kvp {

bool lba_range_len(uint64_t set_size, uint64_t kv_size, uint64_t sector, uint64_t* n_sectors) {
  if (sector == 0) return false;
  const unsigned __int128 bytes = static_cast<unsigned __int128>(set_size) * kv_size;
  const unsigned __int128 n = (bytes + (sector - 1)) / sector;
  if (n >> 64) return false;
  *n_sectors = static_cast<uint64_t>(n);
  return true;
}

// ---- io_uring with raw system calls ----------------------------------------------------------------------------------
bool Uring::open(unsigned entries) {
  close();
  io_uring_params prm;
  memset(&prm, 0, sizeof prm);
  fd_ = static_cast<int>(syscall(__NR_io_uring_setup, entries, &prm));
  if (fd_ < 0) { fd_ = -1; return false; }
  entries_ = prm.sq_entries;
  sq_ring_bytes_ = prm.sq_off.array + prm.sq_entries * sizeof(unsigned);
  cq_ring_bytes_ = prm.cq_off.cqes + prm.cq_entries * sizeof(io_uring_cqe);
  const bool single = prm.features & IORING_FEAT_SINGLE_MMAP;
  if (single) sq_ring_bytes_ = cq_ring_bytes_ = std::max(sq_ring_bytes_, cq_ring_bytes_);
  sq_ring_ = mmap(nullptr, sq_ring_bytes_, PROT_READ | PROT_WRITE, MAP_SHARED | MAP_POPULATE, fd_, IORING_OFF_SQ_RING);
  cq_ring_ = single ? sq_ring_ : mmap(nullptr, cq_ring_bytes_, PROT_READ | PROT_WRITE, MAP_SHARED | MAP_POPULATE, fd_, IORING_OFF_CQ_RING);
  sqes_bytes_ = prm.sq_entries * sizeof(io_uring_sqe);
  sqes_ = mmap(nullptr, sqes_bytes_, PROT_READ | PROT_WRITE, MAP_SHARED | MAP_POPULATE, fd_, IORING_OFF_SQES);
  if (sq_ring_ == MAP_FAILED || cq_ring_ == MAP_FAILED || sqes_ == MAP_FAILED) {
    if (sq_ring_ == MAP_FAILED) sq_ring_ = nullptr;
    if (cq_ring_ == MAP_FAILED) cq_ring_ = nullptr;
    if (sqes_ == MAP_FAILED) sqes_ = nullptr;
    close();
    return false;
  }
  auto at = [](void* base, unsigned off) { return reinterpret_cast<unsigned*>(static_cast<char*>(base) + off); };
  sq_head_ = at(sq_ring_, prm.sq_off.head);
  sq_tail_ = at(sq_ring_, prm.sq_off.tail);
  sq_mask_ = at(sq_ring_, prm.sq_off.ring_mask);
  sq_array_ = at(sq_ring_, prm.sq_off.array);
  cq_head_ = at(cq_ring_, prm.cq_off.head);
  cq_tail_ = at(cq_ring_, prm.cq_off.tail);
  cq_mask_ = at(cq_ring_, prm.cq_off.ring_mask);
  cqes_ = static_cast<char*>(cq_ring_) + prm.cq_off.cqes;
  to_submit_ = 0;
  return true;
}

void Uring::close() {
  if (sqes_) munmap(sqes_, sqes_bytes_);
  if (cq_ring_ && cq_ring_ != sq_ring_) munmap(cq_ring_, cq_ring_bytes_);
  if (sq_ring_) munmap(sq_ring_, sq_ring_bytes_);
  sqes_ = cq_ring_ = sq_ring_ = nullptr;
  if (fd_ >= 0) ::close(fd_);
  fd_ = -1;
}

bool Uring::queue(bool write, int file, void* buf, uint32_t len, uint64_t off, uint64_t user_data) {
  const unsigned tail = *sq_tail_, head = __atomic_load_n(sq_head_, __ATOMIC_ACQUIRE);
  if (tail - head >= entries_) return false;
  const unsigned idx = tail & *sq_mask_;
  io_uring_sqe* e = static_cast<io_uring_sqe*>(sqes_) + idx;
  memset(e, 0, sizeof *e);
  e->opcode = write ? IORING_OP_WRITE : IORING_OP_READ;
  e->fd = file;
  e->off = off;
  e->addr = reinterpret_cast<uint64_t>(buf);
  e->len = len;
  e->user_data = user_data;
  sq_array_[idx] = idx;
  __atomic_store_n(sq_tail_, tail + 1, __ATOMIC_RELEASE);
  ++to_submit_;
  return true;
}

unsigned Uring::drop_unsubmitted() {
  const unsigned n = to_submit_;
  __atomic_store_n(sq_tail_, *sq_tail_ - n, __ATOMIC_RELEASE);  // no SQPOLL: the kernel reads the tail only inside io_uring_enter
  to_submit_ = 0;
  return n;
}

int Uring::flush() {
  while (to_submit_) {
    const long r = syscall(__NR_io_uring_enter, fd_, to_submit_, 0, 0, nullptr, 0);
    if (r < 0) {
      if (errno == EINTR || errno == EAGAIN || errno == EBUSY) continue;
      return errno;
    }
    to_submit_ -= static_cast<unsigned>(r);
  }
  return 0;
}

bool Uring::reap(uint64_t* user_data, int32_t* res) {
  const unsigned head = *cq_head_;
  if (head == __atomic_load_n(cq_tail_, __ATOMIC_ACQUIRE)) return false;
  const io_uring_cqe* c = static_cast<const io_uring_cqe*>(cqes_) + (head & *cq_mask_);
  *user_data = c->user_data;
  *res = c->res;
  __atomic_store_n(cq_head_, head + 1, __ATOMIC_RELEASE);
  return true;
}

int Uring::wait_one() {
  for (;;) {
    const long r = syscall(__NR_io_uring_enter, fd_, 0, 1, IORING_ENTER_GETEVENTS, nullptr, 0);
    if (r >= 0) return 0;
    if (errno != EINTR) return errno;
  }
}

// ---- the device ------------------------------------------------------------------------------------------------------
int SsdDevice::open(const char* path, uint64_t capacity, uint32_t sector, std::string* err) {
  close();
  if (!path || !*path) { *err = "an SSD-type pool device needs a path (block device or file)"; return KVPOOL_EINVAL; }
  if (sector && (sector < 512 || sector > 65536 || (sector & (sector - 1)))) { *err = "sector_bytes must be a power of two in 512..65536"; return KVPOOL_EINVAL; }
  struct stat st {};
  const bool exists = ::stat(path, &st) == 0;
  blockdev_ = exists && S_ISBLK(st.st_mode);
  if (exists && !blockdev_ && !S_ISREG(st.st_mode)) { *err = std::string(path) + " is neither a block device nor a regular file"; return KVPOOL_EINVAL; }
  const int base = O_RDWR | O_CLOEXEC | (blockdev_ ? 0 : O_CREAT);
  direct_ = true;
  fd_ = ::open(path, base | O_DIRECT, 0600);
  if (fd_ < 0 && errno == EINVAL) {  // the file system has no direct I/O (some tmpfs / overlay set-ups): buffered, and say so
    direct_ = false;
    fd_ = ::open(path, base, 0600);
  }
  if (fd_ < 0) { *err = std::string("open ") + path + ": " + strerror(errno); return KVPOOL_EIO; }
  path_ = path;
  created_ = !exists;
  uint64_t size = 0;
  if (blockdev_) {
    int ssz = 0;
    if (ioctl(fd_, BLKGETSIZE64, &size) != 0 || ioctl(fd_, BLKSSZGET, &ssz) != 0 || ssz <= 0) { *err = std::string("ioctl ") + path + ": " + strerror(errno); close(); return KVPOOL_EIO; }
    if (sector == 0) sector = static_cast<uint32_t>(ssz);
    if (sector % static_cast<uint32_t>(ssz)) { *err = "sector_bytes is not a multiple of the device's logical sector size " + std::to_string(ssz); close(); return KVPOOL_EINVAL; }
    if (capacity > size) { *err = "capacity exceeds the block device (" + std::to_string(size) + " bytes)"; close(); return KVPOOL_EINVAL; }
  } else {
    if (sector == 0) sector = 4096;
    if (fstat(fd_, &st) != 0) { *err = std::string("fstat: ") + strerror(errno); close(); return KVPOOL_EIO; }
    if (static_cast<uint64_t>(st.st_size) < capacity && ftruncate(fd_, static_cast<off_t>(capacity)) != 0) {
      *err = std::string("ftruncate ") + path + ": " + strerror(errno);
      close();
      return KVPOOL_EIO;
    }
  }
  sector_ = sector;
  capacity_ = capacity / sector * sector;
  if (capacity_ == 0) { *err = "capacity below one sector"; close(); return KVPOOL_EINVAL; }
  edge_ = static_cast<uint8_t*>(aligned_alloc(4096, std::max<uint32_t>(sector_, 4096)));
  if (!edge_) { *err = "out of memory"; close(); return KVPOOL_ENOMEM; }
  if (direct_) {  // does the file system take direct I/O at this sector size?  (a 4 KiB-sector file system refuses 512-byte requests)
    if (::pread(fd_, edge_, sector_, 0) < 0 && errno == EINVAL) {
      const int fl = fcntl(fd_, F_GETFL);
      if (fl < 0 || fcntl(fd_, F_SETFL, fl & ~O_DIRECT) != 0) { *err = std::string("direct I/O refused at ") + std::to_string(sector_) + "-byte sectors"; close(); return KVPOOL_EIO; }
      direct_ = false;
    }
  }
  return KVPOOL_OK;
}

void SsdDevice::close() {
  stop();
  if (fd_ >= 0) ::close(fd_);
  fd_ = -1;
  if (created_ && !path_.empty()) ::unlink(path_.c_str());  // a stand-in file this device created goes away with it
  created_ = false;
  path_.clear();
  free(edge_);
  edge_ = nullptr;
}

void SsdDevice::start(uint32_t n_lanes, uint64_t lane_bytes, uint8_t* const bounce[2], volatile uint32_t* const gpu_seq[2],
                      volatile uint32_t* const cpu_seq[2], uint32_t stride) {
  stop();
  n_lanes_ = n_lanes;
  lane_bytes_ = lane_bytes;
  stride_ = stride;
  for (int d = 0; d < 2; ++d) { bounce_[d] = bounce[d]; gpu_seq_[d] = gpu_seq[d]; cpu_seq_[d] = cpu_seq[d]; }
  stopping_ = false;
  const char* sync = getenv("KVPOOL_SSD_SYNC");
  depth_ = 1;
  if (!(sync && *sync == '1') && ring_.open(std::max(8u, 4 * n_lanes))) depth_ = std::max(2u, 2 * n_lanes);
  worker_ = depth_ > 1 ? std::thread([this] { run_async(); }) : std::thread([this] { run(); });
}

void SsdDevice::stop() {
  if (!worker_.joinable()) return;
  drain();
  {
    std::lock_guard<std::mutex> l(mu_);
    stopping_ = true;
  }
  cv_.notify_all();
  worker_.join();
  ring_.close();
}

void SsdDevice::submit(const SsdCmd& c) {
  {
    std::lock_guard<std::mutex> l(mu_);
    q_.push_back(c);
    ++submitted_;
  }
  cv_.notify_one();
}

void SsdDevice::drain() {
  std::unique_lock<std::mutex> l(mu_);
  cv_done_.wait(l, [this] { return finished_ == submitted_; });
}

// Poll for the GPU's half of a command (the paper polls NVMe completions on a dedicated core; here the
// worker polls the flag a stream write-value raises): spin briefly, then poll every 20 us.  Gives up only when the pool says
// the GPU is gone (abort(), from kvpool_destroy after a failed device synchronize) — never by the clock: a stream that is
// legitimately held up (long work in front of it, an external event) hands its lane over late, and a command that had
// given up by then would leave the layer marked as stored with nothing written.
bool SsdDevice::wait_flag(const volatile uint32_t* f, uint32_t v) {
  for (int i = 0; i < 4096; ++i) {
    if (seq_reached(f, v)) return true;
    __builtin_ia32_pause();
  }
  const timespec nap{0, 20000};
  for (;;) {
    if (seq_reached(f, v)) return true;
    if (abort_.load(std::memory_order_relaxed)) return false;
    nanosleep(&nap, nullptr);
  }
}

int SsdDevice::rw_full(bool write, uint64_t off, uint8_t* buf, uint64_t n) {
  while (n) {
    const ssize_t r = write ? ::pwrite(fd_, buf, n, static_cast<off_t>(off)) : ::pread(fd_, buf, n, static_cast<off_t>(off));
    if (r < 0) {
      if (errno == EINTR) continue;
      return errno;
    }
    if (r == 0) return EIO;  // end of device inside an allocated range
    buf += r;
    off += static_cast<uint64_t>(r);
    n -= static_cast<uint64_t>(r);
  }
  return 0;
}

bool SsdDevice::gpu_half_arrived(const SsdCmd& c) const {
  const int d = c.op == SsdCmd::kWrite ? 1 : 0;
  const volatile uint32_t* gpu = gpu_seq_[d] + static_cast<uint64_t>(c.lane) * stride_;
  // a store needs the GPU's copy into the lane (gpu_seq >= use); a retrieve needs the lane drained of its previous use
  return seq_reached(gpu, c.op == SsdCmd::kWrite ? c.use : c.use - 1);
}

int SsdDevice::prepare_store(const SsdCmd& c) {
  uint8_t* const buf = bounce_[1] + static_cast<uint64_t>(c.lane) * lane_bytes_;
  const uint64_t body = c.head + c.len, total = (body + sector_ - 1) / sector_ * sector_;
  int e = 0;
  if (c.head) {  // the range starts inside a sector that holds a neighbour's bytes: keep them
    e = rw_full(false, c.file_off, edge_, sector_);
    if (!e) memcpy(buf, edge_, c.head);
  }
  if (!e && total > body) {
    if (c.zero_tail) memset(buf + body, 0, total - body);
    else {
      e = rw_full(false, c.file_off + total - sector_, edge_, sector_);
      if (!e) memcpy(buf + body, edge_ + (sector_ - (total - body)), total - body);
    }
  }
  return e;
}

void SsdDevice::complete(const SsdCmd& c, int e, bool lane_is_ours) {
  const int d = c.op == SsdCmd::kWrite ? 1 : 0;
  if (e) {
    int none = 0;
    error_.compare_exchange_strong(none, e);
    failed_.fetch_add(1);
    // A failed retrieve still hands its lane over (no stream may wait for ever), and the unpack kernel then scatters
    // whatever the lane holds into the caller's paged KV.  The lanes are shared by all requests and keep their last
    // contents, so that must not be the lane as it stands: the caller gets zeroes, never another request's KV.  (Not when
    // the GPU's half never arrived — the GPU is gone, and its previous kernel may formally still own the lane.)
    if (d == 0 && lane_is_ours)
      memset(bounce_[0] + static_cast<uint64_t>(c.lane) * lane_bytes_, 0, static_cast<size_t>(std::min<uint64_t>(c.head + c.len, lane_bytes_)));
  }
  // the hand-over completes even on failure: no stream waits for ever
  __atomic_store_n(cpu_seq_[d] + static_cast<uint64_t>(c.lane) * stride_, c.use, __ATOMIC_RELEASE);
  done_[d].fetch_add(1);
}

void SsdDevice::execute(const SsdCmd& c) {
  const int d = c.op == SsdCmd::kWrite ? 1 : 0;
  uint8_t* const buf = bounce_[d] + static_cast<uint64_t>(c.lane) * lane_bytes_;
  volatile uint32_t* const gpu = gpu_seq_[d] + static_cast<uint64_t>(c.lane) * stride_;
  const uint64_t body = c.head + c.len, total = (body + sector_ - 1) / sector_ * sector_;
  int e = 0;
  if (total > lane_bytes_ || c.file_off % sector_ || c.file_off + total > capacity_) e = EINVAL;
  // SSD_Direct_Retrieve: the lane is free once the GPU has drained its previous use; read the LBA range into it.
  // SSD_Direct_Store: wait for the GPU's copy into the lane, complete the first / last sector, write the LBA range.
  bool ours = true;
  if (!wait_flag(gpu, c.op == SsdCmd::kWrite ? c.use : c.use - 1)) { ours = false; e = e ? e : ECANCELED; }
  if (!e && c.op == SsdCmd::kWrite) e = prepare_store(c);
  if (!e) e = rw_full(c.op == SsdCmd::kWrite, c.file_off, buf, total);
  complete(c, e, ours);
}

void SsdDevice::run() {
  for (;;) {
    SsdCmd c;
    {
      std::unique_lock<std::mutex> l(mu_);
      cv_.wait(l, [this] { return stopping_ || !q_.empty(); });
      if (q_.empty()) return;
      c = q_.front();
      q_.pop_front();
    }
    execute(c);
    {
      std::lock_guard<std::mutex> l(mu_);
      ++finished_;
    }
    cv_done_.notify_all();
  }
}

// The asynchronous worker.  Commands leave the queue in submission order into a small window (`depth_`); a command's disk
// I/O is submitted to the ring as soon as the GPU's half has arrived AND no earlier command still in the window touches
// the same sectors with a write on either side (a retrieve after a store of the same range, a store's read-modify-write of
// a sector it shares with its neighbour); completions are reaped from the ring in whatever order the device finishes them.
struct SsdDevice::Active {
  SsdCmd c;
  uint64_t lo, hi;  // byte range of whole sectors the command touches
  uint64_t id;
  enum { kWaiting, kInFlight } state;
};

void SsdDevice::run_async() {
  std::vector<Active> win;
  uint64_t next_id = 1;
  unsigned idle = 0;
  for (;;) {
    bool progress = false;
    {  // take commands off the queue, in order, while the window has room
      std::unique_lock<std::mutex> l(mu_);
      if (win.empty()) {
        cv_.wait(l, [this] { return stopping_ || !q_.empty(); });
        if (q_.empty()) return;
      }
      while (!q_.empty() && win.size() < depth_) {
        Active a;
        a.c = q_.front();
        q_.pop_front();
        const uint64_t total = (a.c.head + a.c.len + sector_ - 1) / sector_ * sector_;
        a.lo = a.c.file_off;
        a.hi = a.c.file_off + total;
        a.id = next_id++;
        a.state = Active::kWaiting;
        win.push_back(a);
        progress = true;
      }
    }
    unsigned finished = 0;
    std::vector<uint64_t> queued;  // ids handed to the ring in this round, in order
    for (size_t k = 0; k < win.size(); ++k) {
      Active& a = win[k];
      if (a.state != Active::kWaiting) continue;
      bool blocked = false;  // an earlier command of the window overlaps and one of the two writes
      for (size_t j = 0; j < k && !blocked; ++j)
        blocked = win[j].lo < a.hi && a.lo < win[j].hi && (win[j].c.op == SsdCmd::kWrite || a.c.op == SsdCmd::kWrite);
      if (blocked) continue;
      int e = 0;
      const uint64_t total = a.hi - a.lo;
      if (!gpu_half_arrived(a.c)) {  // (checked first, so that a command that fails for another reason fails owning its lane)
        if (abort_.load(std::memory_order_relaxed)) e = ECANCELED;  // the GPU is gone; never by the clock (wait_flag)
        else continue;
      }
      const bool ours = e == 0;
      if (!e && (total > lane_bytes_ || a.lo % sector_ || a.hi > capacity_ || total > 0x7fffffffull)) e = EINVAL;
      const int d = a.c.op == SsdCmd::kWrite ? 1 : 0;
      uint8_t* const buf = bounce_[d] + static_cast<uint64_t>(a.c.lane) * lane_bytes_;
      if (!e && d == 1) e = prepare_store(a.c);
      if (!e && !ring_.queue(d == 1, fd_, buf, static_cast<uint32_t>(total), a.lo, a.id)) continue;  // ring full: next round
      progress = true;
      if (e) {
        complete(a.c, e, ours);
        a.id = 0;  // done
        ++finished;
      } else {
        a.state = Active::kInFlight;
        queued.push_back(a.id);
      }
    }
    if (int e = ring_.flush()) {
      // The kernel refused the submission: fail the entries of THIS round it did not accept (the last `left` queued) and take
      // them off the ring.  Commands it accepted, now or in earlier rounds, are on the disk's side: their lanes stay theirs
      // until their completions are reaped.
      const unsigned left = ring_.drop_unsubmitted();
      for (size_t q = queued.size() - std::min<size_t>(left, queued.size()); q < queued.size(); ++q)
        for (auto& a : win)
          if (a.id == queued[q] && a.state == Active::kInFlight) { complete(a.c, e, true); a.id = 0; ++finished; break; }
    }
    uint64_t id;
    int32_t res;
    while (ring_.reap(&id, &res)) {
      progress = true;
      for (auto& a : win) {
        if (a.id != id || a.state != Active::kInFlight) continue;
        int e = res < 0 ? -res : 0;
        const uint64_t total = a.hi - a.lo;
        if (!e && static_cast<uint64_t>(res) < total) {  // short transfer: finish it synchronously
          const int d = a.c.op == SsdCmd::kWrite ? 1 : 0;
          uint8_t* const buf = bounce_[d] + static_cast<uint64_t>(a.c.lane) * lane_bytes_;
          e = res == 0 ? EIO : rw_full(d == 1, a.lo + static_cast<uint64_t>(res), buf + res, total - static_cast<uint64_t>(res));
        }
        complete(a.c, e, true);
        a.id = 0;
        ++finished;
        break;
      }
    }
    if (finished) {
      win.erase(std::remove_if(win.begin(), win.end(), [](const Active& a) { return a.id == 0; }), win.end());
      {
        std::lock_guard<std::mutex> l(mu_);
        finished_ += finished;
      }
      cv_done_.notify_all();
    }
    if (progress) { idle = 0; continue; }
    // nothing moved: every command of the window waits for the GPU or for the disk
    bool waiting_for_gpu = false;
    for (auto& a : win) waiting_for_gpu |= a.state == Active::kWaiting;
    if (!waiting_for_gpu && !win.empty()) { ring_.wait_one(); continue; }  // only the disk: sleep in the kernel until it completes one
    if (++idle < 2048) __builtin_ia32_pause();
    else {
      const timespec nap{0, 20000};
      nanosleep(&nap, nullptr);
    }
  }
}

int SsdDevice::read_bytes(uint64_t off, void* dst, uint64_t n, uint8_t* scratch, uint64_t scratch_bytes) {
  uint8_t* out = static_cast<uint8_t*>(dst);
  while (n) {
    const uint64_t at = off / sector_ * sector_, head = off - at;
    const uint64_t take = std::min(n, scratch_bytes - head);
    const uint64_t total = (head + take + sector_ - 1) / sector_ * sector_;
    const int e = rw_full(false, at, scratch, total);
    if (e) return e;
    memcpy(out, scratch + head, take);
    out += take;
    off += take;
    n -= take;
  }
  return 0;
}

int SsdDevice::io_span(bool write, uint64_t off, uint64_t n, uint8_t* scratch, uint64_t scratch_bytes) {
  while (n) {
    const uint64_t take = std::min(n, scratch_bytes);
    const int e = rw_full(write, off, scratch, (take + sector_ - 1) / sector_ * sector_);
    if (e) return e;
    off += take;
    n -= take;
  }
  return 0;
}

}  // namespace kvp
