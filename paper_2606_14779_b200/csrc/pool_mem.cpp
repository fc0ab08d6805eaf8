// Pinned, GPU-mapped, optionally NUMA-bound host buffers.  libnuma is not in the image, so binding
// uses the raw mbind / move_pages syscalls and /sys/devices/system/node.
#include "pool_mem.hpp"

#include <cuda_runtime.h>
#include <dirent.h>
#include <errno.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <sys/mman.h>
#include <sys/syscall.h>
#include <unistd.h>
#include <sched.h>

#include <algorithm>
#include <thread>
#include <vector>

#include "../../include/kvpool.h"

namespace kvp {

constexpr uint64_t kHugePage = 2ull << 20;

int numa_node_count() {
  int n = 0;
  if (DIR* d = opendir("/sys/devices/system/node")) {
    while (dirent* e = readdir(d))
      if (strncmp(e->d_name, "node", 4) == 0 && e->d_name[4] >= '0' && e->d_name[4] <= '9') ++n;
    closedir(d);
  }
  return n > 0 ? n : 1;
}

// NUMA node the GPU's PCIe root port hangs off, from sysfs; -1 when unknown (single-node boxes report -1 or 0).
int gpu_numa_node(int cuda_device) {
  char bdf[32] = {0};
  if (cudaDeviceGetPCIBusId(bdf, sizeof(bdf), cuda_device) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  for (char* c = bdf; *c; ++c)
    if (*c >= 'A' && *c <= 'F') *c = static_cast<char>(*c - 'A' + 'a');  // sysfs spells the address in lower case
  const std::string path = std::string("/sys/bus/pci/devices/") + bdf + "/numa_node";
  FILE* f = fopen(path.c_str(), "r");
  if (!f) return -1;
  int node = -1;
  if (fscanf(f, "%d", &node) != 1) node = -1;
  fclose(f);
  return node >= 0 && node < numa_node_count() ? node : -1;
}

static int query_node(void* page) {
  int status = -1;
  void* pages[1] = {page};
  if (syscall(SYS_move_pages, 0, 1ul, pages, nullptr, &status, 0) != 0) return -1;
  return status >= 0 ? status : -1;
}

// First touch of [m, m+bytes) by up to 16 threads (one 4 KiB page at a time; with transparent huge pages every
// 512th touch faults a whole 2 MiB page in).  Page zeroing is what pinning a large buffer costs: on the B200 box
// one thread faults 2.6 GB/s of 4 KiB pages, 16 threads over huge pages 30+ GB/s.
static void first_touch(char* m, uint64_t bytes) {
  cpu_set_t set;
  unsigned cpus = sched_getaffinity(0, sizeof(set), &set) == 0 ? static_cast<unsigned>(CPU_COUNT(&set)) : 1u;
  uint64_t threads = std::min<uint64_t>(std::min<unsigned>(cpus ? cpus : 1u, 16u), std::max<uint64_t>(bytes >> 26, 1));  // >= 64 MiB each
  const uint64_t chunk = ((bytes + threads - 1) / threads + kHugePage - 1) / kHugePage * kHugePage;
  auto touch = [m, bytes, chunk](uint64_t k) {
    const uint64_t hi = std::min(bytes, (k + 1) * chunk);
    for (uint64_t off = k * chunk; off < hi; off += 4096) reinterpret_cast<volatile char*>(m)[off] = 0;
  };
  std::vector<std::thread> pool;
  for (uint64_t k = 1; k < threads; ++k) {
    try { pool.emplace_back(touch, k); }
    catch (...) { touch(k); }  // no thread to be had: this one does the chunk
  }
  touch(0);
  for (auto& t : pool) t.join();
}

// Host memory a new buffer can still take: MemAvailable, capped by the cgroup's limit where there is one.  Faulting in
// more than that would wake the OOM killer instead of failing the call, so registered_alloc refuses first.
static uint64_t read_u64_after(const char* path, const char* key) {
  FILE* f = fopen(path, "r");
  if (!f) return ~0ull;
  char line[256];
  uint64_t v = ~0ull;
  while (fgets(line, sizeof(line), f)) {
    if (key) {
      if (strncmp(line, key, strlen(key)) == 0) { v = strtoull(line + strlen(key), nullptr, 10); break; }
    } else {
      if (line[0] >= '0' && line[0] <= '9') v = strtoull(line, nullptr, 10);  // "max" stays ~0
      break;
    }
  }
  fclose(f);
  return v;
}

uint64_t available_host_bytes() {
  uint64_t avail = read_u64_after("/proc/meminfo", "MemAvailable:");
  if (avail != ~0ull) avail *= 1024;  // kB
  const uint64_t cg_max = read_u64_after("/sys/fs/cgroup/memory.max", nullptr);
  const uint64_t cg_cur = read_u64_after("/sys/fs/cgroup/memory.current", nullptr);
  if (cg_max != ~0ull && cg_cur != ~0ull) avail = std::min(avail, cg_max > cg_cur ? cg_max - cg_cur : 0);
  return avail;
}

// mmap (2 MiB aligned, MADV_HUGEPAGE) + optional mbind + parallel first touch + cudaHostRegister.  Returns KVPOOL_OK,
// or a code with *err set and nothing left allocated.
static int registered_alloc(HostBuffer* hb, uint64_t bytes, int bind_node, bool strict_numa, std::string* err) {
  const uint64_t avail = available_host_bytes();
  if (avail != ~0ull && bytes > avail) {
    *err = "host memory: " + std::to_string(bytes) + " bytes wanted, " + std::to_string(avail) + " available";
    return KVPOOL_ENOMEM;
  }
  const uint64_t span = bytes + kHugePage;
  void* raw = mmap(nullptr, span, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS | MAP_NORESERVE, -1, 0);
  if (raw == MAP_FAILED) { *err = std::string("mmap: ") + strerror(errno); return KVPOOL_ENOMEM; }
  char* m = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(raw) + kHugePage - 1) & ~static_cast<uintptr_t>(kHugePage - 1));
  madvise(m, bytes, MADV_HUGEPAGE);  // advisory: without THP the buffer is made of 4 KiB pages, still touched in parallel
  if (bind_node >= 0) {
    unsigned long mask[16] = {0};
    mask[bind_node / 64] = 1ul << (bind_node % 64);
    const long rc = syscall(SYS_mbind, m, bytes, 2 /*MPOL_BIND*/, mask, sizeof(mask) * 8, 0);
    if (rc != 0 && strict_numa) {
      *err = std::string("mbind: ") + strerror(errno);
      munmap(raw, span);
      return KVPOOL_ENUMA;
    }
  }
  first_touch(m, bytes);  // the pages exist (on the bound node) before they are pinned
  const cudaError_t e = cudaHostRegister(m, bytes, cudaHostRegisterMapped | cudaHostRegisterPortable);
  if (e != cudaSuccess) {
    cudaGetLastError();
    *err = std::string("cudaHostRegister: ") + cudaGetErrorString(e);
    munmap(raw, span);
    return e == cudaErrorMemoryAllocation ? KVPOOL_ENOMEM : KVPOOL_ECUDA;
  }
  hb->host = m;
  hb->map_base = raw;
  hb->map_bytes = span;
  hb->registered = true;
  return KVPOOL_OK;
}

int host_buffer_alloc(HostBuffer* hb, uint64_t bytes, int numa_node, bool write_combined, bool strict_numa, bool cuda_hostalloc,
                      std::string* err) {
  *hb = HostBuffer{};
  hb->bytes = bytes;
  hb->numa_requested = numa_node;
  bool want_bind = numa_node >= 0;
  if (want_bind && numa_node >= numa_node_count()) {
    if (strict_numa) { *err = "NUMA node " + std::to_string(numa_node) + " does not exist"; return KVPOOL_ENUMA; }
    want_bind = false;  // fall back to first-touch placement; numa_actual reports where the pages landed
  }
  // Default: pages this library faults in itself (huge, in parallel) and then registers — an order of magnitude faster
  // to create than cudaHostAlloc for the tens of GiB a pool holds, identical on the link.  cudaHostAlloc serves
  // write-combined buffers, callers that ask for it, and boxes where registration is refused (no NUMA request pending).
  int rc = KVPOOL_ECUDA;
  if (!write_combined && !(cuda_hostalloc && !want_bind)) {
    rc = registered_alloc(hb, bytes, want_bind ? numa_node : -1, strict_numa, err);
    if (rc == KVPOOL_ENUMA || rc == KVPOOL_ENOMEM) return rc;  // strict binding refused / no room; a refused registration falls back to cudaHostAlloc
  }
  if (rc != KVPOOL_OK) {
    unsigned flags = cudaHostAllocMapped | cudaHostAllocPortable | (write_combined ? cudaHostAllocWriteCombined : 0);
    void* m = nullptr;
    const cudaError_t e = cudaHostAlloc(&m, bytes, flags);
    if (e != cudaSuccess) {
      cudaGetLastError();
      *err = std::string("cudaHostAlloc: ") + cudaGetErrorString(e);
      return e == cudaErrorMemoryAllocation ? KVPOOL_ENOMEM : KVPOOL_ECUDA;
    }
    hb->host = m;
  }
  const cudaError_t e = cudaHostGetDevicePointer(&hb->dev_alias, hb->host, 0);
  if (e != cudaSuccess) {
    *err = std::string("cudaHostGetDevicePointer: ") + cudaGetErrorString(e);
    host_buffer_free(hb);
    return KVPOOL_ECUDA;
  }
  hb->numa_actual = write_combined ? -1 : query_node(hb->host);
  return KVPOOL_OK;
}

int device_buffer_alloc(HostBuffer* hb, uint64_t bytes, int gpu, int pool_gpu, std::string* err) {
  *hb = HostBuffer{};
  hb->bytes = bytes;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || gpu < 0 || gpu >= ndev) {
    cudaGetLastError();
    *err = "GPU " + std::to_string(gpu) + " does not exist";
    return KVPOOL_EINVAL;
  }
  if (gpu != pool_gpu) {
    int can = 0;
    cudaError_t e = cudaDeviceCanAccessPeer(&can, pool_gpu, gpu);
    if (e != cudaSuccess || !can) {
      cudaGetLastError();
      *err = "GPU " + std::to_string(pool_gpu) + " cannot access GPU " + std::to_string(gpu) + " as a peer";
      return KVPOOL_ECUDA;
    }
    e = cudaDeviceEnablePeerAccess(gpu, 0);  // current device is pool_gpu
    if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) {
      *err = std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e);
      return KVPOOL_ECUDA;
    }
    cudaGetLastError();
    cudaSetDevice(gpu);
  }
  void* m = nullptr;
  const cudaError_t e = cudaMalloc(&m, bytes);
  if (gpu != pool_gpu) cudaSetDevice(pool_gpu);
  if (e != cudaSuccess) {
    cudaGetLastError();
    *err = std::string("cudaMalloc: ") + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? KVPOOL_ENOMEM : KVPOOL_ECUDA;
  }
  hb->dev_alias = m;
  hb->gpu = gpu;
  return KVPOOL_OK;
}

void host_buffer_free(HostBuffer* hb) {
  if (hb->gpu >= 0) {
    if (hb->dev_alias) cudaFree(hb->dev_alias);  // UVA: cudaFree finds the owning device
    *hb = HostBuffer{};
    return;
  }
  if (!hb->host) return;
  if (hb->registered) {
    cudaHostUnregister(hb->host);
    munmap(hb->map_base, hb->map_bytes);
  } else {
    cudaFreeHost(hb->host);
  }
  *hb = HostBuffer{};
}

}  // namespace kvp
