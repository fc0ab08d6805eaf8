// Pool-device buffers: pinned, GPU-mapped, optionally NUMA-bound host memory (the MEM type of PAPER.md:132, 155), or
// device memory of the pool's GPU / an NVLink peer (the HBM type).
#pragma once
#include <cstdint>
#include <string>

namespace kvp {

struct HostBuffer {
  void* host = nullptr;      // CPU address; nullptr for an HBM-type buffer
  void* dev_alias = nullptr; // address the pool's GPU uses for the bytes (MEM: UVA alias of host; HBM: the device pointer)
  int gpu = -1;              // HBM type: CUDA ordinal that holds the buffer; -1 = MEM type
  uint64_t bytes = 0;
  int numa_requested = -1;
  int numa_actual = -1;      // node of the first page after touching, -1 if it cannot be queried
  bool registered = false;   // true: mmap + cudaHostRegister; false: cudaHostAlloc
  void* map_base = nullptr;  // registered: the mapping that holds `host` (2 MiB-aligned inside it) and its length
  uint64_t map_bytes = 0;
};

// Returns 0 or a KVPOOL_E* code and fills err.  strict_numa: fail instead of falling back when the
// pages cannot be bound to numa_node.  cuda_hostalloc: take the buffer from cudaHostAlloc instead of faulting huge
// pages in in parallel and registering them (kept for comparison; a NUMA request still goes through mbind + register).
int host_buffer_alloc(HostBuffer* hb, uint64_t bytes, int numa_node, bool write_combined, bool strict_numa, bool cuda_hostalloc,
                      std::string* err);
// HBM-type buffer: cudaMalloc on `gpu`, peer access enabled from `pool_gpu` when they differ.  The current device is
// `pool_gpu` on entry and on return.
int device_buffer_alloc(HostBuffer* hb, uint64_t bytes, int gpu, int pool_gpu, std::string* err);
void host_buffer_free(HostBuffer* hb);
int numa_node_count();
uint64_t available_host_bytes();  // MemAvailable capped by the cgroup limit; ~0 when unknown
int gpu_numa_node(int cuda_device);  // -1 when sysfs does not say

}  // namespace kvp
