// Pinned, GPU-mapped, optionally NUMA-bound host buffers: the MEM-type pool devices.
#pragma once
#include <cstdint>
#include <string>

namespace kvp {

struct HostBuffer {
  void* host = nullptr;      // CPU address
  void* dev_alias = nullptr; // address the GPU uses for the same bytes (UVA: normally equal to host)
  uint64_t bytes = 0;
  int numa_requested = -1;
  int numa_actual = -1;      // node of the first page after touching, -1 if it cannot be queried
  bool registered = false;   // true: mmap + cudaHostRegister; false: cudaHostAlloc
};

// Returns 0 or a KVPOOL_E* code and fills err.  strict_numa: fail instead of falling back when the
// pages cannot be bound to numa_node.
int host_buffer_alloc(HostBuffer* hb, uint64_t bytes, int numa_node, bool write_combined, bool strict_numa, std::string* err);
void host_buffer_free(HostBuffer* hb);
int numa_node_count();

}  // namespace kvp
