// sm_100a pack / unpack kernels for paged KV blocks.
//
// Pure data movement: no tensor cores.  Two variants of the same gather/scatter, both templated on the
// direction, both usable with a device staging buffer (HBM-bound) or with mapped pinned host stripes on
// the pool side (host-link-bound, "zero-copy"):
//
//   kv_copy_vec16 : every warp moves 4 KiB pieces with 8 x 16-byte ld.global.nc.L1::no_allocate per lane
//                   issued back to back, then 8 x st.global.L1::no_allocate — 512 contiguous bytes per
//                   warp instruction, 128 B per lane in flight.
//   kv_copy_bulk  : one elected lane per warp drives a ring of shared-memory stages with
//                   cp.async.bulk global->shared (mbarrier complete_tx) and cp.async.bulk shared->global
//                   (bulk groups); whole chunks of a block move without touching registers.
//
// Addressing of unit j is described in kernels.cuh (LayerArgs).
#include "kernels.cuh"

#include <utility>

#include "../../include/kvpool.h"

namespace kvp {
namespace {

constexpr int kVecMaxThreads = 512;
constexpr uint32_t kBulkBarrierBytes = 1024;          // in front of the ring: 512 B of mbarriers (warps*stages <= 64), 512 B of destination pointers

__device__ __forceinline__ int4 ld_stream(const void* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(void* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}

// Profiling: the launch's own execution span on the device clock.  Every CTA (vec16) or issuing warp (bulk) folds its
// start and its end — the last CTAs after their stores are globally visible — into {min, max}; event pairs around a launch also count whatever the
// stream's front end adds (notably under a concurrent copy-engine stream).
__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void span_begin(unsigned long long* span) {
  if (span) atomicMin(span, global_ns());
}
__device__ __forceinline__ void span_end(unsigned long long* span) {
  if (span) atomicMax(span + 1, global_ns());
}

// Programmatic dependent launch (sm_90+): a launch that carries cudaLaunchAttributeProgrammaticStreamSerialization may
// start while the kernel before it on the stream is still running.  Every kernel here lets its successor go at once
// (launch_dependents: the successor's CTAs become resident, set up their barriers and indices) and touches global memory
// only after griddep_wait(), which returns once the predecessor grid has completed and its writes are visible.  Without
// the launch attribute both instructions do nothing.  What it buys: the launch latency and the pipeline ramp of layer
// l+1's kernel hide under layer l's kernel when an engine issues one small zero-copy launch per layer.
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// The three orderings of kernels.cuh (kChain*).
__device__ __forceinline__ void chain_enter(uint32_t chain) {
  if (chain == kChainHead) {
    griddep_wait();
    griddep_launch_dependents();
  } else {
    griddep_launch_dependents();
    if (chain != kChainFollower) griddep_wait();
  }
}
__device__ __forceinline__ void chain_exit(uint32_t chain) {
  if (chain == kChainFollower) griddep_wait();
}

// Decode work item t of a layer split into `pieces` pieces per K (or V) block of `piece_bytes` bytes.
struct Piece {
  uint8_t* paged;
  uint8_t* pooled;
  uint32_t bytes;
  uint32_t layer;  // MultiArgs: index of the piece's layer in the launch
};
// Table check (opt-in, kvpool_set_table_check): a table entry outside the paged pool must neither be read nor written.
// The piece is turned into a copy of the pool-side bytes onto themselves (harmless in both directions, and the bulk ring
// keeps its load/store rhythm); the entry is counted once, by the lane that handles the first piece of its K block.
__device__ __forceinline__ void reject(Piece& p, unsigned long long* bad, bool first_piece) {
  p.paged = p.pooled;
  if (first_piece && (threadIdx.x & 31u) == 0 && bad) atomicAdd(bad, 1ull);
}

// A piece is decoded in two steps, so that a caller that knows its next piece early (the single issuing lane of the bulk
// kernel) can have the table reads in flight while it waits for something else: decode_load issues the global loads for
// piece r of unit `local` and does no arithmetic on their results; decode_finish turns them into addresses.
struct RawPiece {
  int32_t phys;
  uint32_t d, s, r;
  uint32_t layer;  // MultiArgs only
};
__device__ __forceinline__ RawPiece decode_load(const LayerArgs& a, uint32_t local, uint32_t r) {
  RawPiece m;
  uint32_t j;
  if (a.order) {  // device-major chunk: unit `local` of one device's slot range (uniform across the launch)
    j = __ldg(a.order + a.j0 + local);
    m.d = 0;
    m.s = local;
  } else {
    j = a.visit ? __ldg(a.visit + a.j0 + local) : a.j0 + local;
    m.d = __ldg(a.dev + j);
    m.s = __ldg(a.slot + j);
  }
  m.phys = __ldg(a.table + j);
  m.r = r;
  m.layer = 0;
  return m;
}
template <bool CHECK = true>
__device__ __forceinline__ Piece decode_finish(const LayerArgs& a, const RawPiece& m, uint32_t pieces, uint32_t piece_bytes) {
  const uint32_t half = m.r >= pieces ? 1u : 0u;  // 0: K block, 1: V block
  const uint32_t off = (m.r - half * pieces) * piece_bytes;
  Piece p;
  p.paged = (half ? a.v_base : a.k_base) + static_cast<uint64_t>(m.phys) * a.stride + off;
  p.pooled = reinterpret_cast<uint8_t*>(a.pool_base[m.d]) + (static_cast<uint64_t>(m.s) * 2u + half) * a.kvb + off;
  p.bytes = min(piece_bytes, a.kvb - off);
  p.layer = 0;
  if constexpr (CHECK)
    if (a.nphys_check && static_cast<uint32_t>(m.phys) >= a.nphys_check) reject(p, a.bad, m.r == 0);
  return p;
}

__device__ __forceinline__ RawPiece decode_load(const MultiArgs& a, uint32_t unit, uint32_t r) {
  uint32_t lo = 0, hi = a.n;  // last layer with first_unit <= unit
  while (hi - lo > 1) {
    const uint32_t mid = (lo + hi) >> 1;
    if (a.d[mid].first_unit <= unit) lo = mid;
    else hi = mid;
  }
  const MultiDesc& L = a.d[lo];
  const uint32_t j = unit - L.first_unit;
  RawPiece m;
  m.phys = __ldg(L.table + j);
  m.d = __ldg(L.dev + j);
  m.s = __ldg(L.slot + j);
  m.r = r;
  m.layer = lo;
  return m;
}
template <bool CHECK = true>
__device__ __forceinline__ Piece decode_finish(const MultiArgs& a, const RawPiece& m, uint32_t pieces, uint32_t piece_bytes) {
  const MultiDesc& L = a.d[m.layer];
  const uint32_t half = m.r >= pieces ? 1u : 0u;
  const uint32_t off = (m.r - half * pieces) * piece_bytes;
  Piece p;
  p.paged = (half ? L.v_base : L.k_base) + static_cast<uint64_t>(m.phys) * a.stride + off;
  p.pooled = reinterpret_cast<uint8_t*>(__ldg(L.pool_base + m.d) + a.delta[m.d]) + (static_cast<uint64_t>(m.s) * 2u + half) * a.kvb + off;
  p.bytes = min(piece_bytes, a.kvb - off);
  p.layer = m.layer;
  if constexpr (CHECK)
    if (a.nphys_check && static_cast<uint32_t>(m.phys) >= a.nphys_check) reject(p, a.bad, m.r == 0);
  return p;
}

// Work item t of a launch whose K (or V) blocks are split into `pieces` pieces of `piece_bytes` bytes.
template <bool CHECK = true, class Args>
__device__ __forceinline__ Piece decode(const Args& a, uint64_t t, uint32_t pieces, uint32_t piece_bytes) {
  const uint32_t per_unit = 2u * pieces;
  const uint32_t unit = static_cast<uint32_t>(t / per_unit);
  const uint32_t r = static_cast<uint32_t>(t - static_cast<uint64_t>(unit) * per_unit);
  return decode_finish<CHECK>(a, decode_load(a, unit, r), pieces, piece_bytes);
}
__device__ __forceinline__ uint32_t units(const LayerArgs& a) { return a.K; }
__device__ __forceinline__ uint32_t units(const MultiArgs& a) { return a.total_units; }

// SIGNAL (MultiArgs only): per-layer completion flags, see kernels.cuh.
__device__ __forceinline__ void signal_piece(const MultiArgs& a, const Piece& p, uint32_t pieces, uint32_t lane) {
  __threadfence();  // this lane's stores of the piece are visible device-wide ...
  __syncwarp();     // ... and so are the other lanes' before lane 0 counts the piece
  if (lane != 0) return;
  const uint32_t want = a.d[p.layer].K * 2u * pieces;
  if (atomicAdd(a.sig_count + p.layer, 1u) + 1u == want) {
    a.sig_count[p.layer] = 0;  // clean for the next launch that is given this set of flags
    __threadfence();
    atomicExch(a.sig_flag + p.layer, a.sig_seq);
  }
}

template <bool PACK, int kVecUnroll, class Args, bool SIGNAL = false>
__global__ void __launch_bounds__(kVecMaxThreads) kv_copy_vec16(const __grid_constant__ Args a) {
  constexpr uint32_t kVecPiece = kVecUnroll * 32 * 16;  // bytes per warp iteration (4 KiB at unroll 8)
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t warps_per_cta = blockDim.x >> 5;
  const uint64_t nwarps = static_cast<uint64_t>(gridDim.x) * warps_per_cta;
  const uint32_t pieces = (a.kvb + kVecPiece - 1) / kVecPiece;
  const uint64_t total = static_cast<uint64_t>(units(a)) * 2u * pieces;
  chain_enter(a.chain);
  if (threadIdx.x == 0) span_begin(a.span);
  for (uint64_t t = static_cast<uint64_t>(blockIdx.x) * warps_per_cta + (threadIdx.x >> 5); t < total; t += nwarps) {
    const Piece p = decode(a, t, pieces, kVecPiece);
    const uint8_t* src = (PACK ? p.paged : p.pooled) + lane * 16u;
    uint8_t* dst = (PACK ? p.pooled : p.paged) + lane * 16u;
    int4 v[kVecUnroll];
    if (p.bytes == kVecPiece) {
#pragma unroll
      for (int u = 0; u < kVecUnroll; ++u) v[u] = ld_stream(src + u * 512);
#pragma unroll
      for (int u = 0; u < kVecUnroll; ++u) st_stream(dst + u * 512, v[u]);
    } else {  // ragged last piece of a block (kvb not a multiple of 4 KiB; always a multiple of 16)
#pragma unroll
      for (int u = 0; u < kVecUnroll; ++u)
        if (u * 512u + lane * 16u < p.bytes) v[u] = ld_stream(src + u * 512);
#pragma unroll
      for (int u = 0; u < kVecUnroll; ++u)
        if (u * 512u + lane * 16u < p.bytes) st_stream(dst + u * 512, v[u]);
    }
    if constexpr (SIGNAL) signal_piece(a, p, pieces, lane);
  }
  if (a.span) {  // uniform across the grid
    // The end of the launch is set by the CTAs that retire last; only those wait for their stores to land (a fence in
    // every CTA keeps each one resident for a store round trip longer: +3 us on an 80 us launch of 8 waves).
    if (gridDim.x - blockIdx.x <= 512u) __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) span_end(a.span);
  }
  chain_exit(a.chain);
}

// ---- cp.async.bulk / mbarrier primitives (PTX ISA 8.x, sm_90+; SASS: UBLKCP, SYNCS) ------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "KV_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra KV_DONE_%=;\n"
      "bra KV_WAIT_%=;\n"
      "KV_DONE_%=:\n"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read_1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Each warp's lane 0 owns `stages` shared-memory buffers of `chunk` bytes and walks its share of the
// layer's chunks: up to stages-1 loads are in flight while the oldest landed chunk is stored out.
// CHECK: compiled with the opt-in table check (the single issuing lane is latency-bound: the unchecked build keeps the
// check's compare and branch out of its loop — 2 % on an HBM-bound launch).
template <bool PACK, class Args, bool CHECK>
__global__ void __launch_bounds__(256) kv_copy_bulk(const __grid_constant__ Args a, uint32_t chunk, uint32_t stages) {
  extern __shared__ __align__(128) uint8_t smem[];
  if ((threadIdx.x & 31u) != 0) return;
  const uint32_t warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const uint32_t bar0 = smem_u32(smem) + warp * stages * 8u;
  const uint32_t buf0 = smem_u32(smem) + kBulkBarrierBytes + warp * stages * chunk;
  if (a.chain != kChainHead) griddep_launch_dependents();
  for (uint32_t s = 0; s < stages; ++s) mbar_init(bar0 + 8u * s, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  if (a.chain != kChainFollower) griddep_wait();
  if (a.chain == kChainHead) griddep_launch_dependents();
  span_begin(a.span);

  const uint32_t pieces = a.kvb / chunk;  // host guarantees chunk | kvb
  const uint32_t per_unit = 2u * pieces;
  const uint64_t total = static_cast<uint64_t>(units(a)) * per_unit;
  const uint64_t gw = static_cast<uint64_t>(blockIdx.x) * nw + warp, ngw = static_cast<uint64_t>(gridDim.x) * nw;
  const uint64_t mine = gw < total ? (total - gw + ngw - 1) / ngw : 0;

  // The lane is the only issue slot of its ring, so nothing slow may sit between two of its cp.async.bulk: its pieces
  // gw, gw + ngw, ... are walked as (unit, piece in unit) with a carry (no division in the loop), stage indices and the
  // barrier parity are counters, the stages' destinations sit in shared memory, and the table reads of the NEXT piece are
  // issued before the lane goes to wait for the oldest load, so that they have landed when it comes back to issue.
  uint32_t unit = static_cast<uint32_t>(gw / per_unit), r = static_cast<uint32_t>(gw % per_unit);
  const uint32_t du = static_cast<uint32_t>(ngw / per_unit), dr = static_cast<uint32_t>(ngw % per_unit);
  auto advance = [&] {
    unit += du;
    r += dr;
    if (r >= per_unit) { r -= per_unit; ++unit; }
  };
  uint8_t** const out_ring = reinterpret_cast<uint8_t**>(smem + kBulkBarrierBytes / 2) + warp * stages;  // destination of the chunk in each stage
  uint32_t s_issue = 0;
  auto issue = [&](const RawPiece& m) {
    const Piece p = decode_finish<CHECK>(a, m, pieces, chunk);
    out_ring[s_issue] = PACK ? p.pooled : p.paged;
    mbar_arrive_expect_tx(bar0 + 8u * s_issue, chunk);
    bulk_g2s(buf0 + s_issue * chunk, PACK ? p.paged : p.pooled, chunk, bar0 + 8u * s_issue);
    if (++s_issue == stages) s_issue = 0;
  };
  uint64_t issued = 0;
  RawPiece next{};
  if (mine) next = decode_load(a, unit, r);
  while (issued < mine && issued + 1 < stages) {
    const RawPiece cur = next;
    ++issued;
    advance();
    if (issued < mine) next = decode_load(a, unit, r);
    issue(cur);
  }
  uint32_t s_cons = 0, parity = 0;
  for (uint64_t i = 0; i < mine; ++i) {
    mbar_wait(bar0 + 8u * s_cons, parity);
    bulk_s2g(out_ring[s_cons], buf0 + s_cons * chunk, chunk);
    bulk_commit();
    if (++s_cons == stages) { s_cons = 0; parity ^= 1u; }
    if (issued < mine) {
      bulk_wait_read_1();  // the store issued one iteration ago has drained its stage: refill that stage
      const RawPiece cur = next;
      ++issued;
      advance();
      if (issued < mine) next = decode_load(a, unit, r);
      issue(cur);
    }
  }
  bulk_wait_all();
  span_end(a.span);
  chain_exit(a.chain);
}

// ---- consumer stand-in: position-weighted 64-bit checksum of the blocks named by a table ---------------------------
__global__ void __launch_bounds__(256) kv_checksum(const uint8_t* __restrict__ k_base, const uint8_t* __restrict__ v_base, uint64_t stride,
                                                   const int32_t* __restrict__ table, uint32_t n_blocks, uint32_t kvb,
                                                   unsigned long long* __restrict__ out) {
  constexpr uint32_t kUnroll = 4, kPiece = kUnroll * 512;   // 2 KiB per warp iteration, 16 B per lane per load
  const uint32_t lane = threadIdx.x & 31u, warps_per_cta = blockDim.x >> 5;
  const uint64_t nwarps = static_cast<uint64_t>(gridDim.x) * warps_per_cta;
  const uint32_t pieces = (kvb + kPiece - 1) / kPiece, words_per_half = kvb / 8;
  const uint64_t total = static_cast<uint64_t>(n_blocks) * 2u * pieces;
  unsigned long long acc = 0;
  for (uint64_t t = static_cast<uint64_t>(blockIdx.x) * warps_per_cta + (threadIdx.x >> 5); t < total; t += nwarps) {
    const uint32_t j = static_cast<uint32_t>(t / (2u * pieces));
    const uint32_t r = static_cast<uint32_t>(t - static_cast<uint64_t>(j) * 2u * pieces);
    const uint32_t half = r >= pieces ? 1u : 0u, c = r - half * pieces;
    const uint8_t* src = (half ? v_base : k_base) + static_cast<uint64_t>(__ldg(table + j)) * stride + c * kPiece + lane * 16u;
    const uint32_t left = kvb - c * kPiece;
    const uint64_t idx0 = (static_cast<uint64_t>(j) * 2u + half) * words_per_half + (c * kPiece + lane * 16u) / 8u;
    int4 v[kUnroll];
#pragma unroll
    for (uint32_t u = 0; u < kUnroll; ++u)
      if (u * 512u + lane * 16u < left) v[u] = ld_stream(src + u * 512u);
#pragma unroll
    for (uint32_t u = 0; u < kUnroll; ++u)
      if (u * 512u + lane * 16u < left) {
        const unsigned long long w0 = (static_cast<unsigned long long>(static_cast<uint32_t>(v[u].y)) << 32) | static_cast<uint32_t>(v[u].x);
        const unsigned long long w1 = (static_cast<unsigned long long>(static_cast<uint32_t>(v[u].w)) << 32) | static_cast<uint32_t>(v[u].z);
        const unsigned long long idx = idx0 + u * 64u;
        acc += w0 * (2ull * idx + 1ull) + w1 * (2ull * idx + 3ull);
      }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0 && acc != 0) atomicAdd(out, acc);
}

__global__ void kv_spin(uint64_t ns) {
  uint64_t t0, t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  do {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  } while (t - t0 < ns);
}

uint32_t bulk_chunk_for(uint32_t kvb, uint32_t want) {
  uint32_t c = 16;
  while (c * 2 <= want && kvb % (c * 2) == 0) c *= 2;
  return c;
}

}  // namespace

template <bool PACK, class Args, bool CHECK>
static cudaError_t bulk_opt_in() {
  return cudaFuncSetAttribute(kv_copy_bulk<PACK, Args, CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

cudaError_t kernels_init() {
  cudaError_t e = bulk_opt_in<true, LayerArgs, false>();
  if (e == cudaSuccess) e = bulk_opt_in<false, LayerArgs, false>();
  if (e == cudaSuccess) e = bulk_opt_in<true, MultiArgs, false>();
  if (e == cudaSuccess) e = bulk_opt_in<false, MultiArgs, false>();
  if (e == cudaSuccess) e = bulk_opt_in<true, LayerArgs, true>();
  if (e == cudaSuccess) e = bulk_opt_in<false, LayerArgs, true>();
  if (e == cudaSuccess) e = bulk_opt_in<true, MultiArgs, true>();
  if (e == cudaSuccess) e = bulk_opt_in<false, MultiArgs, true>();
  return e;
}

cudaError_t launch_checksum(const uint8_t* k_base, const uint8_t* v_base, uint64_t stride, const int32_t* table, uint32_t n_blocks,
                            uint32_t kvb, unsigned long long* out, uint32_t ctas, cudaStream_t stream) {
  if (n_blocks == 0) return cudaSuccess;
  const uint64_t total = static_cast<uint64_t>(n_blocks) * 2u * ((kvb + 2047u) / 2048u);
  const uint64_t want = (total + 7) / 8;
  kv_checksum<<<static_cast<uint32_t>(want < ctas ? want : ctas), 256, 0, stream>>>(k_base, v_base, stride, table, n_blocks, kvb, out);
  return cudaGetLastError();
}

cudaError_t launch_spin(uint64_t ns, cudaStream_t stream) {
  kv_spin<<<1, 1, 0, stream>>>(ns);
  return cudaGetLastError();
}

// One launch, optionally as a programmatic dependent of the kernel before it on the stream.
template <class... Params, class... Given>
static cudaError_t launch_ex(void (*kernel)(Params...), uint32_t grid, uint32_t block, size_t smem, cudaStream_t stream, bool pdl,
                             Given&&... args) {
  cudaLaunchConfig_t c{};
  c.gridDim = dim3(grid);
  c.blockDim = dim3(block);
  c.dynamicSmemBytes = smem;
  c.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  c.attrs = at;
  c.numAttrs = pdl ? 1u : 0u;
  return cudaLaunchKernelEx(&c, kernel, std::forward<Given>(args)...);
}

template <class Args>
static cudaError_t launch_copy(const Args& a, uint32_t n_units, bool pack, const LaunchCfg& cfg, cudaStream_t stream) {
  if (n_units == 0) return cudaSuccess;
  if (cfg.kernel == KVPOOL_KERNEL_BULK) {
    const uint32_t chunk = bulk_chunk_for(a.kvb, cfg.bulk_chunk);
    const uint32_t stages = cfg.bulk_stages < 2 ? 2 : (cfg.bulk_stages > 8 ? 8 : cfg.bulk_stages);
    uint32_t warps = cfg.bulk_warps < 1 ? 1 : (cfg.bulk_warps > 8 ? 8 : cfg.bulk_warps);
    while (warps > 1 && static_cast<uint64_t>(warps) * stages * chunk + kBulkBarrierBytes > 200u * 1024u) --warps;
    const uint64_t total = static_cast<uint64_t>(n_units) * 2u * (a.kvb / chunk);
    const uint64_t want = (total + warps - 1) / warps;
    const size_t smem = kBulkBarrierBytes + static_cast<size_t>(warps) * stages * chunk;
    // persistent ring: never launch more CTAs than are co-resident (shared memory bounds CTAs per SM)
    const uint64_t per_sm = (227u * 1024u) / (smem + 1024u) ? (227u * 1024u) / (smem + 1024u) : 1;
    const uint64_t resident = static_cast<uint64_t>(cfg.sm_count ? cfg.sm_count : 148u) * (per_sm > 32 ? 32 : per_sm);
    uint64_t cap = cfg.ctas < resident ? cfg.ctas : resident;
    const uint32_t grid = static_cast<uint32_t>(want < cap ? want : cap);
    if (a.nphys_check) {
      if (pack) return launch_ex(kv_copy_bulk<true, Args, true>, grid, warps * 32, smem, stream, cfg.pdl, a, chunk, stages);
      return launch_ex(kv_copy_bulk<false, Args, true>, grid, warps * 32, smem, stream, cfg.pdl, a, chunk, stages);
    }
    if (pack) return launch_ex(kv_copy_bulk<true, Args, false>, grid, warps * 32, smem, stream, cfg.pdl, a, chunk, stages);
    return launch_ex(kv_copy_bulk<false, Args, false>, grid, warps * 32, smem, stream, cfg.pdl, a, chunk, stages);
  } else {
    const uint32_t unroll = cfg.vec_unroll == 4 ? 4 : (cfg.vec_unroll == 16 ? 16 : 8);
    const uint32_t threads = cfg.vec_threads ? cfg.vec_threads : kVecMaxThreads;
    const uint32_t piece = unroll * 512;
    const uint32_t pieces = (a.kvb + piece - 1) / piece;
    const uint64_t total = static_cast<uint64_t>(n_units) * 2u * pieces;
    const uint64_t want = (total + (threads / 32) - 1) / (threads / 32);
    const uint32_t grid = static_cast<uint32_t>(want < cfg.ctas ? want : cfg.ctas);
#define KV_LAUNCH_VEC(U)                                                                                          \
  (pack ? launch_ex(kv_copy_vec16<true, U, Args>, grid, threads, 0, stream, cfg.pdl, a)                           \
        : launch_ex(kv_copy_vec16<false, U, Args>, grid, threads, 0, stream, cfg.pdl, a))
    if (unroll == 4) return KV_LAUNCH_VEC(4);
    if (unroll == 16) return KV_LAUNCH_VEC(16);
    return KV_LAUNCH_VEC(8);
#undef KV_LAUNCH_VEC
  }
}

cudaError_t launch_layer_copy(const LayerArgs& a, bool pack, const LaunchCfg& cfg, cudaStream_t stream) {
  return launch_copy(a, a.K, pack, cfg, stream);
}

// A retrieve that raises a flag per layer (MultiArgs::sig_flag): the 16-byte kernel, whose stores are plain and can be
// fenced piece by piece (the bulk kernel's asynchronous stores retire in groups).
static cudaError_t launch_multi_signal(const MultiArgs& a, const LaunchCfg& cfg, cudaStream_t stream) {
  if (a.total_units == 0) return cudaSuccess;
  const uint32_t threads = cfg.vec_threads ? cfg.vec_threads : kVecMaxThreads;
  const uint32_t pieces = (a.kvb + 4095u) / 4096u;
  const uint64_t total = static_cast<uint64_t>(a.total_units) * 2u * pieces;
  const uint64_t want = (total + (threads / 32) - 1) / (threads / 32);
  const uint32_t grid = static_cast<uint32_t>(want < cfg.ctas ? want : cfg.ctas);
  return launch_ex(kv_copy_vec16<false, 8, MultiArgs, true>, grid, threads, 0, stream, cfg.pdl, a);
}

cudaError_t launch_multi_copy(const MultiArgs& a, bool pack, const LaunchCfg& cfg, cudaStream_t stream) {
  if (a.sig_flag && !pack) return launch_multi_signal(a, cfg, stream);
  return launch_copy(a, a.total_units, pack, cfg, stream);
}

}  // namespace kvp
