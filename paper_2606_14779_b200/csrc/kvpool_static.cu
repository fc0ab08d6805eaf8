// libkvpool.so: kvpool_pack_static — the in-device pack (a5) for callers that must not allocate GPU memory.
//
// Who that is: a serving engine normally hands nearly all of HBM to its own paged-KV allocator at start-up, so a
// cudaMalloc made later from its decode loop can simply fail; and even when it succeeds, cudaMalloc / cudaFree wait for
// the whole device, which stalls every stream of the engine for the length of the call.  Plug-ins that run inside such
// an engine (a KV connector called per layer, say) are in the same position.  The pooled path of this library keeps its
// placement maps — dev[j] and slot[j] of every logical block, Algorithm 1 l.13-16 — in device memory that kvpool_place
// takes from cudaMalloc.  This file gives those callers the gather kernel without any of that: the two maps live in ONE
// file-scope __device__ array of fixed size, a small kernel fills them on the GPU (the closed form of the weighted
// round-robin, one thread per block), and the library's ordinary 16-byte gather kernel then reads them from there.
//
// What follows from the array being static:
//   - it costs kStaticBytes (160 KiB) of HBM on every GPU that loads the library, until the process exits;
//   - a layer of more than KVPOOL_STATIC_MAX_BLOCKS blocks does not fit and is refused (EINVAL), never truncated;
//   - every call on a GPU uses the same array.  Calls issued to ONE stream follow each other and are safe; two calls
//     whose kernels can overlap on the GPU (different streams, no event between them) race on it and corrupt each
//     other's output.  Nothing in it has to start at zero: the map kernel rewrites entries [0, K) before the gather
//     reads them, and entries at K and beyond (the last call's) are never read.
//   - in host code the array's NAME is only a stand-in the runtime uses to find the device-side object; it is not an
//     address a kernel may be given.  The address comes from cudaGetSymbolAddress, asked once per GPU with that GPU
//     current (scratch_of below), and that is what the kernels receive.
#include <mutex>

#include "kvpool_internal.hpp"

using namespace kvp;

namespace {

constexpr uint32_t kStaticMax = KVPOOL_STATIC_MAX_BLOCKS;
constexpr size_t kStaticBytes = static_cast<size_t>(kStaticMax) * 5;  // slot[] as uint32, then dev[] as uint8
constexpr int kStaticMaxGpus = 64;

static __device__ __align__(256) uint8_t g_static_scratch[kStaticBytes];

struct StaticCounts {  // c_i of Eq. 2 and the first stage unit of each device's stripe (exclusive prefix sum)
  uint32_t n;
  uint32_t c[KVPOOL_MAX_DEVICES];
  uint32_t start[KVPOOL_MAX_DEVICES];
};

// Thread t handles unit t of the packed buffer = the k-th block (1-based) of device i, and finds the logical block that
// lands there: its rank among all (k / c_i, i) pairs (placement.hpp).  Every entry of [0, K) is written exactly once.
__global__ void __launch_bounds__(256) kv_static_map(const __grid_constant__ StaticCounts p, uint32_t K, uint32_t* __restrict__ slot,
                                                     uint8_t* __restrict__ dev) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= K) return;
  uint32_t i = 0;
  while (i + 1 < p.n && t >= p.start[i] + p.c[i]) ++i;
  const uint64_t ci = p.c[i], k = t - p.start[i] + 1;
  uint64_t pos = k - 1;
  for (uint32_t o = 0; o < p.n; ++o) {
    if (o == i || p.c[o] == 0) continue;
    const uint64_t x = k * p.c[o];  // < 2^64: k <= c_i < 2^32
    pos += (o < i) ? x / ci : (x - 1) / ci;
  }
  slot[pos] = static_cast<uint32_t>(k - 1);
  dev[pos] = static_cast<uint8_t>(i);
}

struct StaticGpu {
  uint8_t* scratch = nullptr;  // device address of g_static_scratch on this GPU
  int sm_count = 0;
};
std::mutex g_static_lock;
StaticGpu g_static_gpu[kStaticMaxGpus];

// Once per GPU, with that GPU current: ask the runtime where the array lives on it.  (This is also what makes the
// runtime load this file's device code onto the GPU, array included, if it has not done so yet.)
int scratch_of(int cuda_device, StaticGpu* out) {
  std::lock_guard<std::mutex> g(g_static_lock);
  StaticGpu& s = g_static_gpu[cuda_device];
  if (!s.scratch) {
    void* ptr = nullptr;
    int sms = 0;
    CU(cudaGetSymbolAddress(&ptr, g_static_scratch));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device));
    if (!ptr || sms <= 0) return fail(KVPOOL_ECUDA, "pack_static: no device address for the scratch array on GPU %d", cuda_device);
    s.sm_count = sms;
    s.scratch = static_cast<uint8_t*>(ptr);
  }
  *out = s;
  return KVPOOL_OK;
}

}  // namespace

extern "C" int kvpool_pack_static(const uint64_t* w, uint32_t n, const kvpool_geometry* geom, uint32_t K, const void* k_base,
                                  const void* v_base, uint64_t stride, const int32_t* table, void* stage_dev, int cuda_device,
                                  void* cuda_stream) {
  if (!w || !geom) return fail(KVPOOL_EINVAL, "pack_static: null weights or geometry");
  if (n == 0 || n > KVPOOL_MAX_DEVICES) return fail(KVPOOL_EINVAL, "pack_static: %u pool devices (1..%u)", n, KVPOOL_MAX_DEVICES);
  if (K > kStaticMax)
    return fail(KVPOOL_EINVAL, "pack_static: a layer of %u blocks exceeds KVPOOL_STATIC_MAX_BLOCKS = %u, the size of the library's static scratch",
                K, kStaticMax);
  const uint64_t kvb = static_cast<uint64_t>(geom->block_tokens) * geom->n_kv_heads * geom->head_dim * geom->elem_bytes;
  if (kvb == 0 || kvb % 16 || kvb > (1u << 30)) return fail(KVPOOL_EINVAL, "pack_static: a K block of %llu bytes (a multiple of 16 up to 1 GiB)", (unsigned long long)kvb);
  if (cuda_device < 0 || cuda_device >= kStaticMaxGpus) return fail(KVPOOL_EINVAL, "pack_static: CUDA device %d (0..%d)", cuda_device, kStaticMaxGpus - 1);
  unsigned __int128 W = 0;
  for (uint32_t i = 0; i < n; ++i) {
    if (w[i] < 1) return fail(KVPOOL_EINVAL, "pack_static: weight %u is zero", i);
    W += w[i];
  }
  if (K == 0) return KVPOOL_OK;
  if (!k_base || !v_base || !table || !stage_dev) return fail(KVPOOL_EINVAL, "pack_static: null device pointer");
  if ((reinterpret_cast<uintptr_t>(k_base) | reinterpret_cast<uintptr_t>(v_base) | reinterpret_cast<uintptr_t>(stage_dev) | stride) & 15u)
    return fail(KVPOOL_EINVAL, "pack_static: k_base, v_base, stage_dev and the block stride must be multiples of 16");

  // Eq. 2 / Alg. 1 l.4-12 on the stack: floors, then one extra block each for the first K - sum devices in (w desc, index asc) order
  StaticCounts p{};
  p.n = n;
  uint64_t sum = 0;
  for (uint32_t i = 0; i < n; ++i) {
    p.c[i] = static_cast<uint32_t>(static_cast<unsigned __int128>(w[i]) * K / W);
    sum += p.c[i];
  }
  uint32_t order[KVPOOL_MAX_DEVICES];
  for (uint32_t i = 0; i < n; ++i) {  // stable insertion sort, heaviest first
    uint32_t at = i;
    while (at > 0 && w[order[at - 1]] < w[i]) { order[at] = order[at - 1]; --at; }
    order[at] = i;
  }
  for (uint64_t r = 0; r < K - sum; ++r) p.c[order[r]] += 1;
  for (uint32_t i = 0, acc = 0; i < n; ++i) { p.start[i] = acc; acc += p.c[i]; }

  DeviceGuard guard(cuda_device);
  StaticGpu gpu;
  int rc = scratch_of(cuda_device, &gpu);
  if (rc != KVPOOL_OK) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  uint32_t* slot_d = reinterpret_cast<uint32_t*>(gpu.scratch);
  uint8_t* dev_d = gpu.scratch + static_cast<size_t>(kStaticMax) * 4;
  kv_static_map<<<(K + 255u) / 256u, 256, 0, s>>>(p, K, slot_d, dev_d);
  CU(cudaGetLastError());

  LayerArgs a{};
  a.k_base = static_cast<uint8_t*>(const_cast<void*>(k_base));
  a.v_base = static_cast<uint8_t*>(const_cast<void*>(v_base));
  a.stride = stride;
  a.table = table;
  a.dev = dev_d;
  a.slot = slot_d;
  a.K = K;
  a.kvb = static_cast<uint32_t>(kvb);
  for (uint32_t i = 0; i < n; ++i) a.pool_base[i] = reinterpret_cast<uint64_t>(static_cast<uint8_t*>(stage_dev) + static_cast<uint64_t>(p.start[i]) * 2u * kvb);
  LaunchCfg cfg{};
  cfg.kernel = KVPOOL_KERNEL_VEC16;
  cfg.ctas = 16u * static_cast<uint32_t>(gpu.sm_count);
  cfg.vec_threads = 512;
  cfg.vec_unroll = 8;
  cfg.sm_count = static_cast<uint32_t>(gpu.sm_count);
  cfg.pdl = false;  // the gather must see the whole map: plain stream order behind kv_static_map
  CU(launch_layer_copy(a, true, cfg, s));
  return KVPOOL_OK;
}
