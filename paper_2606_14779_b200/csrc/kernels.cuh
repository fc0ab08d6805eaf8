// sm_100a pack / unpack kernels (a5, a8 of DESIGN.md §2; fused with a6/a7 when the pool side is mapped
// host memory).  Launch interface only; kernels.cu has the device code.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace kvp {

constexpr uint32_t kMaxDev = 32;

// One layer's work.  Unit j (logical block j) has
//   paged side : K block = kvb bytes at k_base + table[j]*stride, V block likewise at v_base
//   pool side  : P = 2*kvb bytes (K then V) at pool_base[dev[j]] + slot[j]*P
// pool_base[i] is any address the GPU can reach: a device staging buffer (in-device pack/unpack) or the
// device alias of a mapped pinned host stripe (zero-copy offload/retrieve).
struct LayerArgs {
  uint8_t* k_base;
  uint8_t* v_base;
  uint64_t stride;
  const int32_t* table;
  const uint8_t* dev;
  const uint32_t* slot;
  uint32_t K;    // number of units this launch moves ...
  uint32_t j0;   // ... starting at logical block j0 (table/dev/slot are indexed by j0 + local index)
  // Device-major chunk (staged path, layers larger than a staging slot): when `order` is set the launch moves K
  // consecutive SLOTS of ONE pool device instead of K consecutive logical blocks: unit u is logical block
  // order[j0 + u] (the inverse map of that device, ascending in slot) and its pool side is pool_base[0] + u*P, so the
  // chunk is one contiguous piece of that device's stripe: ONE copy per chunk.  dev / slot are not read.
  const uint32_t* order;
  // Visiting order (mixed pools, whole-layer zero-copy launches): when set, unit u is logical block visit[j0 + u] — a
  // permutation of the layer's blocks that lists the blocks of host-memory devices first, so that the link (the slow
  // resource of such a launch: ~50 GB/s next to ~3 TB/s) is busy from the first CTA on instead of receiving its last
  // pieces when the HBM share is nearly done.  dev / slot are read as usual.
  const uint32_t* visit;
  uint32_t kvb;
  unsigned long long* span;  // profiling only (else null): device {min start, max end} of the launch in %globaltimer ns
  unsigned long long* bad;   // table check only (else null): counts table entries outside [0, nphys_check)
  uint32_t nphys_check;      // 0 = the table is trusted (R12); else entries >= this (or negative) are skipped and counted
  uint32_t chain;            // kChain*: how the launch orders itself against the kernel before it on the stream (below)
  uint64_t pool_base[kMaxDev];
};

// Programmatic dependent launch, three ways (kernels.cu).  kChainNone: let the successor become resident at once, touch
// memory only once the predecessor grid has completed — right for a launch that may depend on anything before it.
// A run of launches that do NOT depend on each other (the layers of one batched retrieve: other stripes, other paged
// tensors) can overlap each launch's first transfers with its predecessor's tail instead: the HEAD of the run waits for
// everything before it and only then lets its successor go; a FOLLOWER starts moving bytes at once — whatever the head
// waited for is complete, and the launches between the head and itself are its independent siblings — and waits for its
// predecessor just before it exits, so that grids still complete in stream order and whatever follows the run sees all of it.
constexpr uint32_t kChainNone = 0, kChainHead = 1, kChainFollower = 2;

// Several layers in one launch (tiny layers: one launch latency and one pipeline ramp for the whole batch).  Units are
// numbered across the batch; layer i owns units [first_unit, first_unit + K).  pool_base points at N device-visible
// stripe addresses in global memory (uploaded once per placement).
constexpr uint32_t kMaxBatch = 64;
struct MultiDesc {
  uint8_t* k_base;
  uint8_t* v_base;
  const int32_t* table;
  const uint8_t* dev;
  const uint32_t* slot;
  const uint64_t* pool_base;
  uint32_t K;
  uint32_t first_unit;
};
struct MultiArgs {
  uint64_t stride;
  uint32_t kvb;
  uint32_t n;            // layers in this launch, <= kMaxBatch
  uint32_t total_units;  // sum of K
  uint32_t chain;        // kChain*, as in LayerArgs
  unsigned long long* span;  // as in LayerArgs
  unsigned long long* bad;   // as in LayerArgs
  uint32_t nphys_check;
  // Per-layer completion signals (retrieve only; null = none): the warp that finishes the last piece of layer i of the launch
  // raises sig_flag[i] = sig_seq once every store of that layer is visible device-wide (sig_count[i] counts the pieces and
  // is left at zero again).  A stream wait-value on the flag then stands where an event record after a launch of that
  // layer alone would: ONE launch moves many small layers and still hands them over one by one (kvpool_retrieve_layers_signal).
  uint32_t sig_seq;
  uint32_t* sig_count;
  uint32_t* sig_flag;
  uint64_t delta[kMaxDev];  // added (mod 2^64) to pool_base[i]: 0 for the mapped host stripes themselves, or the
                            // displacement that maps device i's span of stripes onto its copy in a staging slot
  MultiDesc d[kMaxBatch];
};

struct LaunchCfg {
  uint32_t kernel;       // KVPOOL_KERNEL_VEC16 / KVPOOL_KERNEL_BULK
  uint32_t ctas;         // grid size cap
  uint32_t bulk_chunk, bulk_stages, bulk_warps;
  uint32_t vec_threads, vec_unroll;
  uint32_t sm_count;
  bool pdl;              // launch as a programmatic dependent of the kernel before it on the stream
};

// pack = true: paged -> pool side (offload direction); false: pool side -> paged (retrieve direction).
cudaError_t launch_layer_copy(const LayerArgs& a, bool pack, const LaunchCfg& cfg, cudaStream_t stream);
cudaError_t launch_multi_copy(const MultiArgs& a, bool pack, const LaunchCfg& cfg, cudaStream_t stream);
// Consumer stand-in / integrity check: *out += sum over logical blocks j < n, halves h (0 = K, 1 = V) and 64-bit
// words i of  word * (2*idx + 1)  (mod 2^64),  idx = (j*2 + h)*(kvb/8) + i.  Reads the blocks through the table
// exactly as a decode-attention kernel would (K_l*P bytes of HBM reads); `out` must be zeroed by the caller.
cudaError_t launch_checksum(const uint8_t* k_base, const uint8_t* v_base, uint64_t stride, const int32_t* table, uint32_t n_blocks,
                            uint32_t kvb, unsigned long long* out, uint32_t ctas, cudaStream_t stream);
// One thread spins on %globaltimer for `ns` nanoseconds: a calibrated compute stand-in for pipeline experiments.
cudaError_t launch_spin(uint64_t ns, cudaStream_t stream);
// One-time per-device setup (shared-memory opt-in for the bulk kernels).
cudaError_t kernels_init();

}  // namespace kvp
