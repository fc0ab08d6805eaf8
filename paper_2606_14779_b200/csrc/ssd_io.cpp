// KV-passthrough, host side: see ssd_io.hpp.  SSD_Direct_Store / SSD_Direct_Retrieve of PAPER.md:181-185 with the kernel's
// O_DIRECT block path standing where the paper uses SPDK (no NVMe device and no SPDK in this image: DESIGN.md R19).
#include "ssd_io.hpp"

#include <errno.h>
#include <fcntl.h>
#include <linux/fs.h>
#include <sys/ioctl.h>
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
  worker_ = std::thread([this] { run(); });
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
// worker polls the flag a stream write-value raises): spin briefly, then poll every 20 us.  Gives up when the pool says
// the GPU is gone (abort(), from kvpool_destroy after a failed device synchronize) and, as a backstop, after ten minutes.
bool SsdDevice::wait_flag(const volatile uint32_t* f, uint32_t v) {
  for (int i = 0; i < 4096; ++i) {
    if (seq_reached(f, v)) return true;
    __builtin_ia32_pause();
  }
  const auto t0 = std::chrono::steady_clock::now();
  const timespec nap{0, 20000};
  for (uint64_t n = 0;; ++n) {
    if (seq_reached(f, v)) return true;
    if (abort_.load(std::memory_order_relaxed)) return false;
    nanosleep(&nap, nullptr);
    if ((n & 1023) == 1023 && std::chrono::steady_clock::now() - t0 > std::chrono::minutes(10)) return false;
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

void SsdDevice::execute(const SsdCmd& c) {
  const int d = c.op == SsdCmd::kWrite ? 1 : 0;
  uint8_t* const buf = bounce_[d] + static_cast<uint64_t>(c.lane) * lane_bytes_;
  volatile uint32_t* const gpu = gpu_seq_[d] + static_cast<uint64_t>(c.lane) * stride_;
  volatile uint32_t* const cpu = cpu_seq_[d] + static_cast<uint64_t>(c.lane) * stride_;
  const uint64_t body = c.head + c.len, total = (body + sector_ - 1) / sector_ * sector_;
  int e = 0;
  if (total > lane_bytes_ || c.file_off % sector_ || c.file_off + total > capacity_) e = EINVAL;
  if (c.op == SsdCmd::kRead) {
    // SSD_Direct_Retrieve: the lane is free once the GPU has drained its previous use; read the LBA range into it
    if (!wait_flag(gpu, c.use - 1)) e = e ? e : (abort_.load() ? ECANCELED : ETIMEDOUT);
    if (!e) e = rw_full(false, c.file_off, buf, total);
  } else {
    // SSD_Direct_Store: wait for the GPU's copy into the lane, complete the first / last sector, write the LBA range
    if (!wait_flag(gpu, c.use)) e = e ? e : (abort_.load() ? ECANCELED : ETIMEDOUT);
    if (!e && c.head) {  // the range starts inside a sector that holds a neighbour's bytes: keep them
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
    if (!e) e = rw_full(true, c.file_off, buf, total);
  }
  if (e) {
    int none = 0;
    error_.compare_exchange_strong(none, e);
  }
  __atomic_store_n(cpu, c.use, __ATOMIC_RELEASE);  // the handshake completes even on failure: no stream waits for ever
  done_[d].fetch_add(1);
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
