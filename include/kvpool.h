/*
 * kvpool.h — C ABI of the B200-native unified KV pooling hot path (arxiv 2606.14779).
 *
 * The library moves a request's *paged* KV cache between GPU HBM and a pool of "pool devices" — pinned
 * host buffers (type MEM), block storage addressed by LBA (type SSD, KV-passthrough) and GPU memory of
 * NVLink peers (type HBM) —, assigning each layer's KV blocks to pool devices in proportion to
 * their measured bandwidth (Eq. 1-2; Algorithm 1) and retrieving
 * them through a dense global lookup table (Table I; retrieval).
 *
 * Conventions
 *   - Every function returns KVPOOL_OK (0) or a negative KVPOOL_E* code; kvpool_last_error() gives a
 *     thread-local message for the last failure.  Nothing throws or aborts across the ABI.  A call that
 *     fails with EINVAL / ENOMEM / ESTATE has had no effect.
 *   - "host" / "device" after a pointer says where the memory lives.  The caller owns the paged KV
 *     tensors, block tables and CUDA streams; the library owns pool buffers, staging buffers, its own
 *     streams/events and the per-placement tables.  The library never frees or keeps caller memory
 *     beyond the stream work a call enqueues.
 *   - One "KV cache" of the paper = one paged block of one layer: K block then V block,
 *     P = 2*kvb bytes with kvb = block_tokens*n_kv_heads*head_dim*elem_bytes (R6).
 *   - There is no CPU fallback: without a CUDA device kvpool_create fails with KVPOOL_ECUDA.  The
 *     kvpool_plan_* functions are pure host arithmetic and work anywhere.
 *   - A pool handle may be used from several host threads at once (one per request, say), each with
 *     its own CUDA streams: every call that touches pool state takes the pool's lock, and calls only
 *     enqueue work, so the lock is held for microseconds (kvpool_release, kvpool_synchronize and
 *     kvpool_measure_bandwidth hold it while they wait).  A placement is used by one thread at a time;
 *     kvpool_destroy must not race with any other call.
 */
#ifndef KVPOOL_H
#define KVPOOL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KVPOOL_MAX_DEVICES 32u

#if defined(__GNUC__)
#define KVPOOL_API __attribute__((visibility("default")))
#else
#define KVPOOL_API
#endif

enum {
  KVPOOL_OK = 0,
  KVPOOL_EINVAL = -1, /* bad argument: null pointer, bandwidth <= 0, misaligned base/stride, layer/dev out of range */
  KVPOOL_ENOMEM = -2, /* a pool device has no room for its stripe, or host/device allocation failed */
  KVPOOL_ECUDA = -3,  /* a CUDA runtime call failed (message has the CUDA error string) */
  KVPOOL_ENUMA = -4,  /* KVPOOL_DEV_NUMA_STRICT and the pages could not be bound to the requested node */
  KVPOOL_ESTATE = -5, /* retrieve of a layer that was never offloaded; set_bandwidth while placements are live; ... */
  KVPOOL_ENOENT = -6, /* kvpool_glt_find: no KV cache with that identifier */
  KVPOOL_EIO = -7     /* an SSD-type pool device could not be opened, or a store / retrieve command on it failed */
};

/* pool-device flags */
#define KVPOOL_DEV_WRITE_COMBINED 1u /* cudaHostAllocWriteCombined (GPU-read-mostly; CPU reads become slow) */
#define KVPOOL_DEV_NUMA_STRICT 2u    /* fail with ENUMA instead of falling back when binding is impossible */
#define KVPOOL_DEV_CUDA_HOSTALLOC 8u /* take the buffer from cudaHostAlloc.  Default: the library maps the pages itself (2 MiB
                                        aligned, MADV_HUGEPAGE), faults them in with up to 16 threads and pins them with
                                        cudaHostRegister — ~10x faster to create, same link bandwidth; it falls
                                        back to cudaHostAlloc by itself where registration is refused.                       */
#define KVPOOL_DEV_HBM 4u            /* the pool device is GPU memory, not host memory: HBM of GPU `gpu` — an NVLink / NVSwitch
                                        peer of the pool's GPU, or that GPU itself.  Its stripes are reached
                                        by the kernels directly (peer loads / stores); no staging, no copy engine.            */

#define KVPOOL_DEV_SSD 16u           /* the pool device is block storage addressed by LBA (the paper's SSD type, KV-passthrough,
                                        PAPER.md:179-185): `path` names a block device (/dev/nvme0n1, a partition) or a
                                        file standing in for one.  It is opened O_DIRECT - the kernel's page cache and the
                                        file system's data path are bypassed; on a raw block device there is no file system
                                        at all - and driven by the device's own worker thread through asynchronous store /
                                        retrieve commands (io_uring); the pack / unpack kernels reach the pinned bounce lanes
                                        over the link, and GPU streams and the worker hand lanes to each other with stream
                                        write-value / wait-value operations: no copy engine, no host callback, no
                                        synchronisation.  Excludes every other flag.               */

#define KVPOOL_MEASURE_KERNEL_RETRIEVE 2 /* kvpool_measure_bandwidth / kvpool_calibrate `direction`, see there */
#define KVPOOL_MEASURE_KERNEL_OFFLOAD 3

#define KVPOOL_NUMA_AUTO (-2)        /* kvpool_device_desc.numa_node: bind to the NUMA node of the pool's GPU */

/* pool-device types (GLT `type`, Table I) */
enum {
  KVPOOL_TYPE_MEM = 0, /* pinned host memory; location = host pointer                                     */
  KVPOOL_TYPE_SSD = 1, /* block storage (KVPOOL_DEV_SSD); location = logical block address (LBA)          */
  KVPOOL_TYPE_HBM = 2  /* GPU memory (KVPOOL_DEV_HBM); location = device pointer valid on the pool's GPU  */
};

/* transfer paths (kvpool_set_path) */
enum {
  KVPOOL_PATH_AUTO = 0,     /* staged for layers >= the auto threshold, zero-copy below it            */
  KVPOOL_PATH_STAGED = 1,   /* pack/unpack kernel <-> device staging + one cudaMemcpyAsync per stripe  */
  KVPOOL_PATH_ZEROCOPY = 2, /* one kernel reads/writes the mapped host stripes directly over the link  */
  KVPOOL_PATH_HYBRID = 3    /* offload: zero-copy (the kernel's own posted writes, >= 8 CTAs, no staging slot, no copy
                               engine); retrieve: as AUTO.  For engines that evict one request while they fetch another
                               (PAPER.md:166, 241): SM-issued READS collapse under a concurrent GPU->host stream (their
                               128-byte read requests queue behind the write data), SM-issued writes do not, so this is
                               the kernel path that keeps both directions of the link busy — 91 GB/s against 94 staged
                               both ways and 67-74 zero-copy both ways (profiles/r2_duplex.md) — and it leaves the copy
                               engines and the whole staging ring to the retrieve direction                              */
};
/* kernel variants (kvpool_set_tuning) */
enum {
  KVPOOL_KERNEL_VEC16 = 0, /* 16-byte ld.global.nc / st.global, warp-contiguous, unrolled              */
  KVPOOL_KERNEL_BULK = 1   /* cp.async.bulk global->shared->global rings with mbarrier completion      */
};

typedef struct kvpool kvpool_t;                     /* opaque pool                                       */
typedef struct kvpool_placement kvpool_placement_t; /* opaque: one request's GLT + reserved stripes      */

typedef struct {           /* one pool device (Table I)                                    */
  double bandwidth_gbps;   /* b_i of Eq. 1, measured, in 1e9 B/s; > 0                                   */
  uint64_t capacity_bytes; /* size of the buffer the library allocates (pinned + mapped host memory, or */
                           /* device memory with KVPOOL_DEV_HBM), or how much of `path` an SSD-type      */
                           /* device may use; > 0                                                        */
  int32_t numa_node;       /* MEM: -1 = no preference (the pages land on the nodes of the cores that    */
                           /* fault them in: on a multi-socket host prefer KVPOOL_NUMA_AUTO);           */
                           /* KVPOOL_NUMA_AUTO = the node the pool's GPU hangs off (sysfs; no           */
                           /* preference if unknown); else bind the pages to this node                  */
  uint32_t flags;          /* KVPOOL_DEV_*                                                              */
  int32_t gpu;             /* HBM: CUDA ordinal of the GPU that holds the buffer, -1 = the pool's own   */
                           /* GPU; must be peer-accessible from it (ECUDA otherwise).  MEM: ignored     */
  uint32_t link_group;     /* 0 = the device has a transfer resource of its own.  g > 0: it shares one  */
                           /* with every other device of the pool that names the same g - several host  */
                           /* buffers behind one PCIe link, several HBM devices inside one GPU.  Such   */
                           /* devices are served in request order by ONE I/O stream per direction (the  */
                           /* paper's "independent I/O streams", are per independent      */
                           /* resource: copies that share a link only slow each other down, and layer   */
                           /* l+1's copies would delay layer l's), and kvpool_calibrate divides what    */
                           /* they share.  Placement (Eq. 1-2) is untouched: only b_i changes.  An SSD-   */
                           /* type device moves its share on kernel streams of its own, whatever its     */
                           /* group (a stream that waits for a disk must hold up nothing else)           */
  const char* path;        /* SSD: block device or file (host string, copied); NULL otherwise.  The     */
                           /* library owns sectors [0, capacity_bytes / sector_bytes) of it: whatever    */
                           /* they held is overwritten; a file it had to create is removed again by      */
                           /* kvpool_destroy.  Two devices of one pool must not name the same path       */
  uint32_t sector_bytes;   /* SSD: sector size LBAs count in - a power of two in 512..65536 and a       */
                           /* multiple of the device's logical sector; 0 = ask the block device, 4096   */
                           /* for a file.  Otherwise 0                                                  */
  uint32_t reserved;       /* 0                                                                         */
} kvpool_device_desc;

typedef struct { /* geometry of one paged KV block */
  uint32_t n_layers, block_tokens, n_kv_heads, head_dim, elem_bytes;
} kvpool_geometry;

typedef struct {         /* kvpool_set_tuning; 0 in any field = library default                          */
  uint32_t kernel;       /* KVPOOL_KERNEL_* for HBM-bound launches (staged path, kvpool_pack/unpack); always applied */
  uint32_t link_kernel;  /* KVPOOL_KERNEL_* for zero-copy launches (default BULK: 2 CTAs fill the link); always applied */
  uint32_t hbm_ctas;     /* CTAs of an in-device pack/unpack launch (default: a multiple of the SM count) */
  uint32_t link_ctas;    /* CTAs of a zero-copy launch (default 4; profiles/r1_sweep_link.txt)           */
  uint32_t bulk_chunk;   /* bytes per cp.async.bulk (power of two, 1 KiB..32 KiB)                        */
  uint32_t bulk_stages;  /* ring depth per issuing warp                                                 */
  uint32_t bulk_warps;   /* issuing warps per CTA                                                       */
  uint32_t stage_slots;  /* staging buffers in the ring of the staged path (default 2: one fills while the other drains) */
  uint32_t vec_threads;  /* threads per CTA of the vec16 kernel (multiple of 32, 64..512)                */
  uint32_t vec_unroll;   /* 16-byte loads in flight per lane in the vec16 kernel: 4, 8 or 16             */
  uint64_t auto_threshold_bytes; /* PATH_AUTO: layers (or groups) moving fewer bytes than this go zero-copy */
  uint64_t group_bytes;  /* batched calls: consecutive layers are grouped until a group moves at least this much */
  uint64_t stage_chunk_bytes; /* staged path: a staging slot holds at most this much (default 256 MiB, so the ring is at most
                            stage_slots x 256 MiB = 512 MiB of HBM whatever the context length).  A larger layer travels in
                            DEVICE-MAJOR chunks: a chunk is a run of consecutive slots of ONE pool device's stripe, i.e. one
                            contiguous piece of that stripe - ONE cudaMemcpyAsync - gathered / scattered by a launch that finds
                            its logical blocks through the device's inverse map (uploaded with the placement); the copy of
                            chunk c+1 overlaps the pack / unpack of chunk c.  Placement and stripe bytes are the same as
                            without chunking.  UINT64_MAX: no cap (a slot holds the largest layer); at least one block per chunk */
  uint32_t pdl;          /* programmatic dependent launch of the library's kernels (the next layer's launch latency and
                            ramp hide under the current layer's kernel): 1 = on (default), 2 = off                          */
  uint32_t ssd_lanes;    /* SSD-type devices: bounce lanes per device and direction (default 4): a lane is one store /
                            retrieve command in flight - pinned, GPU-mapped host memory: the disk's DMA target on one side,
                            read / written by the pack / unpack kernel over the link on the other                          */
  uint64_t ssd_chunk_bytes; /* SSD-type devices: bytes per command (default 8 MiB; at least one KV cache plus two sectors).
                            ssd_lanes / ssd_chunk_bytes are fixed by the first kvpool_place: ESTATE afterwards           */
} kvpool_tuning;

/* ---- pure host arithmetic (no CUDA, no pool) --------------------------------------------------------
 * Eq. 1: weights.  w_i = floor(b_i*1000 + 0.5) (integer MB/s); p_i = w_i / sum_j w_j exactly.
 * EINVAL if n == 0, n > KVPOOL_MAX_DEVICES or some w_i < 1.                                            */
KVPOOL_API int kvpool_plan_weights(const double* bandwidth_gbps /*host[n]*/, uint32_t n, uint64_t* w_out /*host[n]*/);
/* Eq. 2 / Alg. 1 l.4-16 for one layer of K blocks: counts_out[i] = floor(p_i*K) plus one for the top
 * (K - sum floors) devices by (p_i desc, i asc); dev_out[j], slot_out[j] = smooth weighted round-robin
 * position of logical block j (device, index inside that device's stripe).  dev_out/slot_out may be
 * NULL (counts only).                                                                                  */
KVPOOL_API int kvpool_plan_layer(const uint64_t* w /*host[n]*/, uint32_t n, uint64_t K, uint32_t* counts_out /*host[n]*/,
                      uint8_t* dev_out /*host[K] or NULL*/, uint32_t* slot_out /*host[K] or NULL*/);

/* KV-passthrough: the length, in sectors, of the contiguous LBA range SSD_Direct_Store allocates for an
 * offload set of set_size KV caches of kv_size bytes: ceil(set_size * kv_size / sector_bytes).  EINVAL if sector_bytes
 * is 0 or the result does not fit 64 bits.                                                                          */
KVPOOL_API int kvpool_plan_lba_range(uint64_t set_size, uint64_t kv_size, uint32_t sector_bytes, uint64_t* n_sectors_out /*host*/);

/* The caller's contract on a block table (R12), checked on a HOST copy: K entries, each in [0, nphys), no
 * physical block named twice (a duplicate would make two KV caches race for one block at retrieve).  The hot path
 * never validates tables on the device; engines call this in debug builds or tests.  EINVAL with the first offending
 * entry in kvpool_last_error().  K = 0 is valid.                                                                  */
KVPOOL_API int kvpool_validate_table(const int32_t* table /*host[K]*/, uint64_t K, uint64_t nphys);
/* The same contract checked on the DEVICE, opt-in (hardening / debug builds; compute-sanitizer-free): with nphys > 0
 * every later launch skips table entries outside [0, nphys) — the blocks they name are neither read nor written, so a
 * corrupt table cannot touch another request's KV — and counts them (after an offload the pool slot of a rejected entry
 * holds unspecified bytes).  One compare per 4-16 KiB piece: no measurable
 * cost.  Duplicates are not detected (kvpool_validate_table does that on the host).  nphys = 0 (default) trusts the
 * table.  kvpool_table_errors returns the number of rejected entries of the launches that have completed since the
 * last call and resets it (blocking; the caller synchronises the streams it cares about first).                     */
KVPOOL_API int kvpool_set_table_check(kvpool_t* pool, uint64_t nphys);
KVPOOL_API int kvpool_table_errors(kvpool_t* pool, uint64_t* count_out /*host*/);

/* ---- pool life cycle ----------------------------------------------------------------------------------
 * kvpool_create enumerates the pool devices: allocates one pinned, GPU-mapped host
 * buffer per device (bound to its NUMA node when asked and possible), per-device CUDA streams, events
 * and an empty GLT.  Pins memory — ~10 GB/s of pool on the B200 box (huge pages faulted in by up to 16
 * threads, then cudaHostRegister; KVPOOL_DEV_CUDA_HOSTALLOC: 2.5 GB/s); not on the hot path.
 * cuda_device = CUDA ordinal.                                                                          */
KVPOOL_API int kvpool_create(const kvpool_device_desc* devs /*host[n_devs]*/, uint32_t n_devs, const kvpool_geometry* geom /*host*/,
                  int cuda_device, uint32_t flags /*0*/, kvpool_t** out);
/* Waits for all work the pool enqueued, frees everything including live placements.                    */
KVPOOL_API int kvpool_destroy(kvpool_t* pool);

/* Replace the bandwidths ("measured bandwidth") — ESTATE while any placement is live.     */
KVPOOL_API int kvpool_set_bandwidth(kvpool_t* pool, const double* bandwidth_gbps /*host[n_devs]*/);
/* Measure pool device `dev`: cudaMemcpyAsync of `bytes` (<= capacity) between the pool buffer and a
 * scratch device buffer, `iters` times, median, CUDA events.  direction 0 = pool->GPU (retrieve
 * direction), 1 = GPU->pool.  GB/s counts the bytes moved once (payload), for HBM devices too.  Blocking.
 * direction KVPOOL_MEASURE_KERNEL_RETRIEVE (2) / KVPOOL_MEASURE_KERNEL_OFFLOAD (3): the same bytes moved by the
 * library's own gather / scatter kernel between the device's memory, reached in place (mapped host memory over the
 * link, or HBM), and a scratch paged layout — the rate that counts where the kernels reach the stripes themselves:
 * every device of a pool with HBM-type devices, and the zero-copy path (SM-issued transfers over PCIe run ~8 %
 * below the copy engines).  Measure with the mechanism that will move the bytes.
 * The first `bytes` of the pool buffer are overwritten in either direction (a host buffer measured in
 * direction 0 is first written once by DMA: stripes are always written by an offload before a retrieve
 * reads them, and freshly zeroed pages still held in CPU caches read ~5 % slow until then) — ESTATE
 * while any placement is live.                                                                          */
KVPOOL_API int kvpool_measure_bandwidth(kvpool_t* pool, uint32_t dev, int direction, uint64_t bytes, uint32_t iters, double* gbps_out /*host*/);
/* What each device can count on when the members of a link group run together (pure host arithmetic, no pool):
 * out[i] = alone[i] for link_group[i] == 0, else alone[i] * max_g / sum_g over the members of its group, evaluated
 * left to right in IEEE double - m equal members get 1/m of the shared rate each, unequal members split the best
 * member's rate in proportion to their own, and a group's shares add up to that best rate.  Eq. 1 presumes every
 * device delivers b_i concurrently; bandwidths measured one device at a time over-count devices
 * that share a link.  EINVAL if n == 0, n > KVPOOL_MAX_DEVICES or some alone[i] is not positive and finite.       */
KVPOOL_API int kvpool_share_bandwidth(const double* alone_gbps /*host[n]*/, const uint32_t* link_group /*host[n]*/, uint32_t n,
                           double* out_gbps /*host[n]*/);
/* "Measured bandwidth" of Eq. 1 in one call: kvpool_measure_bandwidth on every pool device in turn
 * (min(bytes, capacity) each), kvpool_share_bandwidth over the pool's link groups, kvpool_set_bandwidth with the
 * result.  bandwidth_out (host[n_devs], may be NULL) receives the installed b_i.  Blocking; ESTATE while any
 * placement is live.                                                                                              */
KVPOOL_API int kvpool_calibrate(kvpool_t* pool, int direction, uint64_t bytes, uint32_t iters, double* bandwidth_out /*host[n_devs]*/);
/* The b_i the pool currently places by (as given to kvpool_create / kvpool_set_bandwidth, or installed by
 * kvpool_calibrate) and each device's link group.  Either out pointer may be NULL.                                */
KVPOOL_API int kvpool_bandwidths(const kvpool_t* pool, double* bandwidth_out /*host[n_devs]*/, uint32_t* link_group_out /*host[n_devs]*/);

KVPOOL_API int kvpool_set_path(kvpool_t* pool, int path /*KVPOOL_PATH_**/);
KVPOOL_API int kvpool_set_tuning(kvpool_t* pool, const kvpool_tuning* t /*host*/);
KVPOOL_API int kvpool_get_tuning(const kvpool_t* pool, kvpool_tuning* t_out /*host*/);

/* Size the staging ring of the staged path now: `stage_slots` device buffers of `bytes` bytes each.  A placement needs
 * max(its largest layer K_l * P, min(group_bytes, all its layers together)) — the second term for the groups of small
 * layers the batched calls form — capped by tune.stage_chunk_bytes when that is set (larger layers then travel in
 * chunks).  kvpool_place grows the ring by itself when a placement needs more, but
 * growing waits for the whole device (cudaDeviceSynchronize) and reallocates; an engine that knows its largest layer
 * calls this once at start-up and no later kvpool_place ever waits for GPU work.  ENOMEM if the device is out of memory. */
KVPOOL_API int kvpool_reserve_staging(kvpool_t* pool, uint64_t bytes);

/* ---- placement: Alg. 1 l.4-16 + stripe allocation + GLT update (a1-a4) ------------------------------
 * blocks_per_layer[l] = K_l, the number of KV blocks of layer l to offload (may differ per layer and
 * may be 0).  Host work plus one upload of the per-layer tables on the library's own stream: the call does not wait for
 * work queued on any other stream, the legacy default stream included (unless the staging ring must grow, see
 * kvpool_reserve_staging).  ENOMEM (nothing reserved) if some pool
 * device cannot hold its stripes.                                                                      */
KVPOOL_API int kvpool_place(kvpool_t* pool, const uint32_t* blocks_per_layer /*host[n_layers]*/, kvpool_placement_t** out);
/* Frees the stripes and tables.  Waits first (host-blocking) for the library's own transfers and for the last work
 * each hot-path call enqueued with this placement on the caller's streams, so the stripes cannot be handed to another
 * request while a kernel still reads or writes them.  (Calls made while a stream was being captured into a CUDA graph
 * are not tracked: a graph that names the placement must not be launched after the release.)  EIO, the placement still
 * live, if a command of an SSD-type device has failed (see kvpool_synchronize): release again to let it go.            */
KVPOOL_API int kvpool_release(kvpool_t* pool, kvpool_placement_t* pl);

/* A request's block tables in ONE upload (a 1K-token request moves 4 MiB per layer: a separate table copy per layer costs
 * more than the layer's own transfer time).  tables_host (host; pageable or pinned; free again when the call returns) is
 * the concatenation, in layer order, of the K_l int32 entries of every layer of the placement — n_entries must equal
 * sum_l K_l; layers with K_l = 0 contribute nothing.  One cudaMemcpyAsync on `stream` into device memory the placement
 * owns.  Afterwards every hot-path call on this placement accepts block_table_dev = NULL (per-layer calls) or
 * block_tables = NULL / NULL entries (batched calls) and then reads the uploaded table of that layer; such a call must be
 * ordered after the upload (same stream, or an event).  May be called again to replace the tables (it then first waits,
 * host-blocking, for the work enqueued with the placement so far).
 * EINVAL on a wrong entry count; entries are not validated (R12).                                          */
KVPOOL_API int kvpool_set_tables(kvpool_t* pool, kvpool_placement_t* pl, const int32_t* tables_host /*host[sum K_l]*/, uint64_t n_entries,
                      void* cuda_stream);

/* ---- the hot path: one layer ---------------------------------------------------------------------------
 * k_base / v_base: device pointers to the layer's K and V planes; physical block p is the kvb bytes at
 * base + p*block_stride_bytes (covers [2,nphys,...] and [nphys,2,...] layouts).  Both bases and the
 * stride must be multiples of 16.  block_table_dev: device int32[K_l], logical -> physical; entries are
 * not validated on the device (duplicates / out-of-range are the caller's contract, R12).
 * Asynchronous: returns once the work is enqueued.
 *
 * kvpool_offload  (Alg. 1 l.17-22, MEMSTORE): gathers the K_l blocks into the N stripes.  Work enqueued
 *   on `stream` after the call may overwrite the source blocks (the gather is ordered on `stream`); the
 *   stripe bytes are complete once kvpool_wait_offloads/kvpool_synchronize says so (zero-copy path: also
 *   ordered on `stream`).  A later kvpool_retrieve of the same layer is ordered after it internally.
 * kvpool_retrieve: scatters the stripes back into the paged layout; complete in
 *   `stream` order.  ESTATE if the layer was never offloaded.  Host->GPU staging copies may run ahead of
 *   `stream` (they touch only library memory), which is what overlaps layer l+1's I/O with layer l's
 *   consumer (layerwise pipelining).                                                       */
KVPOOL_API int kvpool_offload(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, const void* k_base /*device*/,
                   const void* v_base /*device*/, uint64_t block_stride_bytes, const int32_t* block_table_dev,
                   void* cuda_stream);
KVPOOL_API int kvpool_retrieve(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, void* k_base /*device*/, void* v_base /*device*/,
                    uint64_t block_stride_bytes, const int32_t* block_table_dev, void* cuda_stream);
/* Batched forms: layers [first_layer, first_layer + n_layers) in one call, equivalent to the per-layer calls in
 * ascending order provided the paged tensors of different layers do not overlap (the library lets the launches of one
 * call overlap each other's ends).  k_bases / v_bases / block_tables are HOST arrays of n_layers DEVICE pointers (entries of layers
 * with K_l = 0 may be NULL).  Consecutive layers are gathered into groups of at least `group_bytes` (default 64 MiB,
 * at most 64 layers; a large layer travels with the small ones before it) and each group moves as one unit: one
 * fused kernel launch on the zero-copy path, or one pack/unpack launch plus ONE cudaMemcpyAsync per pool device on
 * the staged path (a placement's stripes are contiguous per device across layers).  Small layers thus pay one
 * launch latency and one DMA ramp per group instead of one per layer (1K-token contexts, sliding-window layers).
 * All arguments are validated before anything is enqueued.                                                                            */
KVPOOL_API int kvpool_offload_layers(kvpool_t* pool, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers,
                          const void* const* k_bases /*host[n_layers]*/, const void* const* v_bases /*host[n_layers]*/,
                          uint64_t block_stride_bytes, const int32_t* const* block_tables /*host[n_layers]*/, void* cuda_stream);
KVPOOL_API int kvpool_retrieve_layers(kvpool_t* pool, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers,
                           void* const* k_bases /*host[n_layers]*/, void* const* v_bases /*host[n_layers]*/,
                           uint64_t block_stride_bytes, const int32_t* const* block_tables /*host[n_layers]*/, void* cuda_stream);
/* kvpool_retrieve_layers for a consumer on ANOTHER stream (layerwise pipelining): layer_ready is a HOST
 * array of n_layers caller-owned cudaEvent_t (entries may be NULL); layer_ready[q] is recorded as soon as layer
 * first_layer + q is complete in the paged layout, so the consumer does cudaStreamWaitEvent(consumer, layer_ready[q]) and
 * computes layer q while the pool is still moving layers q+1, ... (the staged path's host->GPU copies run up to
 * `stage_slots` layers ahead).  Layers that travel as one group (small layers, see above) become ready together — except
 * in a request of less than two groups' worth of bytes on KVPOOL_PATH_ZEROCOPY: that one moves as ONE launch
 * whose kernel raises a flag as each layer's last byte lands, and a stream of the library's own turns the flags into the
 * caller's events (stream wait-value, then event record), so every layer is handed over by itself although no launch and
 * no copy is spent on it alone; such events are recorded on that stream, not on `stream`.  (On the other paths such a
 * request is cut into two groups, so that the consumer of the first overlaps the second, and the last eighth of any small
 * request travels as a short group of its own, so that few consumers are left behind the last byte.)  A layer with K_l = 0 is ready
 * at once.  One host call per request instead of one per layer.                                                       */
KVPOOL_API int kvpool_retrieve_layers_signal(kvpool_t* pool, kvpool_placement_t* pl, uint32_t first_layer, uint32_t n_layers,
                                  void* const* k_bases /*host[n_layers]*/, void* const* v_bases /*host[n_layers]*/,
                                  uint64_t block_stride_bytes, const int32_t* const* block_tables /*host[n_layers]*/,
                                  void* const* layer_ready /*host[n_layers] of cudaEvent_t*/, void* cuda_stream);
/* Partial retrieval (prefix reuse, chunked prefetch): like kvpool_retrieve for logical blocks
 * [first_block, first_block + n_blocks) of the layer only.  block_table_dev is still the LAYER's table (indexed by
 * logical block, as at offload); only the entries of the range are read and only their physical blocks written.
 * Because placement is a smooth weighted round-robin (R3), any contiguous range draws on all pool devices
 * in proportion to their bandwidth, within N-1 blocks.  EINVAL if the range exceeds K_l; n_blocks = 0 is a no-op.    */
KVPOOL_API int kvpool_retrieve_range(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, uint32_t first_block, uint32_t n_blocks,
                          void* k_base /*device*/, void* v_base /*device*/, uint64_t block_stride_bytes,
                          const int32_t* block_table_dev, void* cuda_stream);
/* Partial offload — a request's blocks reach the pool in instalments ("at decoding step t, let K(t) denote the set of KV
 * caches that must be offloaded"): like kvpool_offload for logical blocks [first_block, first_block +
 * n_blocks) of the layer only, stored at the places Algorithm 1 gave them when the layer was placed (so the split
 * stays bandwidth-proportional however the layer is cut).  Nothing outside the range's slots is written.  A retrieve
 * (whole or range) needs every block it names to have been offloaded: ESTATE otherwise.  EINVAL if the range exceeds
 * K_l; n_blocks = 0 is a no-op.  kvpool_offload is this call over [0, K_l).                                           */
KVPOOL_API int kvpool_offload_range(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, uint32_t first_block, uint32_t n_blocks,
                         const void* k_base /*device*/, const void* v_base /*device*/, uint64_t block_stride_bytes,
                         const int32_t* block_table_dev /*device[K_l]*/, void* cuda_stream);
/* Make `stream` wait until every offload enqueued so far with `pl` has landed in the pool (on an SSD-type device: until
 * its store commands have been written — a stream wait-value on the flag the device's worker raises).                */
KVPOOL_API int kvpool_wait_offloads(kvpool_t* pool, kvpool_placement_t* pl, void* cuda_stream);
/* Block the host until all work the pool enqueued on its own streams is done (not the caller's), and note which
 * offloads have landed.  After the caller has also synchronised its own streams, later zero-copy calls on those layers
 * enqueue exactly one kernel on `cuda_stream` and nothing else (no event waits or queries), so a zero-copy
 * kvpool_retrieve / kvpool_retrieve_layers / kvpool_retrieve_range can be captured into a CUDA graph and replayed
 * (profiling off; the placement and the tables must outlive the graph).  Also waits for the workers of SSD-type devices;
 * EIO (once) if a store / retrieve command has failed since the last call — the bytes of that command are lost, every
 * hand-over has completed all the same.                                                                             */
KVPOOL_API int kvpool_synchronize(kvpool_t* pool);

/* In-device halves alone (a5 / a8): gather the layer's blocks into `stage_dev` (device, K_l*P bytes) in
 * stripe order — device 0's stripe, then device 1's, ... — or scatter them back from it.  Ordered on
 * `stream`.  These are the kernels whose HBM roofline the bench reports.                                */
KVPOOL_API int kvpool_pack(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, const void* k_base, const void* v_base,
                uint64_t block_stride_bytes, const int32_t* block_table_dev, void* stage_dev, void* cuda_stream);
KVPOOL_API int kvpool_unpack(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, void* k_base, void* v_base,
                  uint64_t block_stride_bytes, const int32_t* block_table_dev, const void* stage_dev, void* cuda_stream);

/* kvpool_pack for callers that must not allocate GPU memory — code running inside a serving engine that has given nearly
 * all of HBM to its own KV allocator (a cudaMalloc made later can fail) and whose decode loop cannot afford the
 * device-wide wait cudaMalloc / cudaFree imply.  No pool, no placement: the call itself works out where Algorithm 1 puts
 * the K blocks of one layer over n pool devices of integer weights w (as from kvpool_plan_weights; Eq. 1-2, Alg. 1
 * l.4-16 — the same counts and the same weighted round-robin as kvpool_plan_layer / kvpool_place) and gathers them into
 * stage_dev (device, K*P bytes, 16-byte aligned) in stripe order, byte for byte what kvpool_pack writes.  The dev / slot
 * maps the gather reads, which kvpool_place keeps in cudaMalloc'd memory, live here in one fixed array inside the
 * library's own device image: 160 KiB of HBM on every GPU that loads the library, held until the process exits.  The call
 * makes no cudaMalloc, cudaFree or other allocating CUDA call; it enqueues two kernels on `cuda_stream` (one fills the
 * maps on the GPU, one gathers) and returns.
 *   - K > KVPOOL_STATIC_MAX_BLOCKS (a 512K-token layer at 16-token blocks): EINVAL, nothing enqueued.  K = 0 is a no-op.
 *   - cuda_device: the CUDA ordinal the pointers and the stream belong to (0..63).  The FIRST call on a GPU also looks up
 *     the array's address on that GPU (and thereby has the runtime load the library's device code there): make that first
 *     call at start-up, before any stream capture.
 *   - All calls on one GPU share the array.  Calls on one stream are ordered and safe.  Calls whose kernels may overlap on
 *     the GPU (different streams with no event between them, or several host threads doing so) RACE on it and give wrong
 *     bytes: order them.  The array keeps the last call's maps; no call depends on what it finds there.
 *   - geom->n_layers is ignored.  EINVAL for n = 0, n > KVPOOL_MAX_DEVICES, a zero weight, a block size or a pointer /
 *     stride that is not a multiple of 16; ECUDA if a CUDA call fails.  The table is not validated (R12).      */
#define KVPOOL_STATIC_MAX_BLOCKS 32768u
KVPOOL_API int kvpool_pack_static(const uint64_t* w /*host[n]*/, uint32_t n, const kvpool_geometry* geom /*host*/, uint32_t K,
                       const void* k_base /*device*/, const void* v_base /*device*/, uint64_t block_stride_bytes,
                       const int32_t* block_table_dev /*device[K]*/, void* stage_dev /*device*/, int cuda_device, void* cuda_stream);

/* ---- introspection (GLT, Table I) -----------------------------------------------------------------------*/
KVPOOL_API int kvpool_n_devices(const kvpool_t* pool, uint32_t* n_out);
KVPOOL_API int kvpool_weights(const kvpool_t* pool, uint64_t* w_out /*host[n_devs]*/);
KVPOOL_API int kvpool_device_info(const kvpool_t* pool, uint32_t dev, void** host_base, uint64_t* capacity_bytes, uint64_t* used_bytes,
                       int32_t* numa_node_actual /* -1 unknown */);
/* Type of pool device `dev` (KVPOOL_TYPE_*) and, for HBM devices, the CUDA ordinal that holds it (-1 for MEM).
 * For an HBM device kvpool_device_info's host_base is NULL.                                              */
KVPOOL_API int kvpool_device_type(const kvpool_t* pool, uint32_t dev, uint32_t* type, int32_t* gpu);
KVPOOL_API int kvpool_counts(const kvpool_placement_t* pl, uint32_t layer, uint32_t* counts_out /*host[n_devs]*/);
/* GLT entry of logical block `block` of `layer`: device_id, type (KVPOOL_TYPE_*), slot inside that device's
 * stripe and the location of its payload (Table I "location"): a host pointer for MEM, a device pointer for HBM. */
KVPOOL_API int kvpool_lookup(const kvpool_placement_t* pl, uint32_t layer, uint32_t block, uint32_t* device_id, uint32_t* type,
                  uint32_t* slot, void** location);
/* Stripe of `layer` on pool device `dev`: its location (host pointer for MEM, device pointer for HBM; NULL when
 * empty) and size.                                                                                              */
KVPOOL_API int kvpool_stripe(const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, void** location, uint64_t* nbytes);
/* Copy the first `nbytes` (<= stripe size) of that stripe into host memory, whatever the device type (memcpy for MEM,
 * blocking cudaMemcpy for HBM).  The caller must have waited for the offload (kvpool_wait_offloads + stream sync).
 * For inspection and tests; not a hot-path call.                                                                 */
KVPOOL_API int kvpool_stripe_read(kvpool_t* pool, const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, void* dst_host, uint64_t nbytes);
/* SSD-type pool devices (GLT `type` = KVPOOL_TYPE_SSD, `location` = LBA; Table I).  For such a device
 * kvpool_stripe returns the first LBA of the stripe's range (cast to a pointer-sized integer) and kvpool_lookup the LBA
 * of the sector in which the KV cache's payload starts; kvpool_device_info's host_base is NULL.
 * kvpool_ssd_range: the contiguous LBA range SSD_Direct_Store allocated for the offload set of (layer, dev):
 *   n_sectors = ceil(c_{l,dev} * P / sector_bytes), first_lba in units of sector_bytes.  The payloads
 *   follow each other in slot order from the first byte of the range; the rest of the last sector is zero.
 * kvpool_ssd_location: where KV cache `block` of `layer` lives: LBA = first_lba + floor(slot*P / sector_bytes) and the
 *   byte inside that sector (0 whenever P is a multiple of the sector size).  EINVAL if the block's device is not SSD.
 * kvpool_ssd_info: sector size, whether the device is open with direct I/O (0 = the file system refused O_DIRECT and
 *   the library fell back to buffered I/O), whether it is a block device (0 = a file standing in for one), and the
 *   store / retrieve commands its worker has completed, and how many commands the worker keeps in flight on the device
 *   (io_uring; 1 = the synchronous fall-back, 0 = no worker yet: it starts with the first kvpool_place or measurement).
 *   Any out pointer may be NULL.                                                                                   */
KVPOOL_API int kvpool_ssd_range(const kvpool_placement_t* pl, uint32_t layer, uint32_t dev, uint64_t* first_lba, uint64_t* n_sectors,
                     uint32_t* sector_bytes);
KVPOOL_API int kvpool_ssd_location(const kvpool_placement_t* pl, uint32_t layer, uint32_t block, uint64_t* lba, uint32_t* byte_in_sector);
KVPOOL_API int kvpool_ssd_info(const kvpool_t* pool, uint32_t dev, uint32_t* sector_bytes, int32_t* direct_io, int32_t* block_device,
                    uint64_t* stores_completed, uint64_t* retrieves_completed, uint32_t* queue_depth);

/* Store / retrieve commands of the pool's SSD-type devices that have failed since kvpool_create (a count that only grows;
 * 0 for a pool without such devices).  Non-blocking and lock-free - it reads the workers' counters - so an engine that
 * pipelines on per-layer events can poll it (before and after a request, say) instead of waiting for the EIO of the next
 * kvpool_synchronize / kvpool_release.  What a failed command leaves behind: a failed RETRIEVE command still hands its
 * bytes over, so that no stream waits for ever and the layer's events fire, but the KV caches it covered arrive as ZERO
 * bytes - never as whatever the shared bounce lane held before, which could be another request's KV; a failed STORE
 * command leaves its LBA range unwritten.  A count that moved while a request was in flight means: do not use that
 * request's KV.                                                                                                      */
KVPOOL_API int kvpool_io_errors(const kvpool_t* pool, uint64_t* failed_out /*host*/);

/* Keyed GLT (Table I `key` = "hash of the KV cache identifier"): give the K_l KV caches of a layer
 * caller-chosen 64-bit identifiers (e.g. the prefix-hash of the tokens a block covers, mixed with the layer), after
 * which any of them is found by identifier alone, across placements — what cross-request prefix reuse needs.
 * kvpool_glt_bind: EINVAL, nothing bound, if an identifier is already bound or repeats.  Identifiers die with their
 * placement (kvpool_release).  kvpool_glt_find returns the Table I fields plus where the entry lives: key (the
 * 64-bit hash the table is indexed by), device_id, type (KVPOOL_TYPE_*), location (pointer of the payload), and the
 * (placement, layer, block) to hand to kvpool_retrieve_range.  Any out pointer may be NULL.  ENOENT if absent.      */
KVPOOL_API int kvpool_glt_bind(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, const uint64_t* ids /*host[K_l]*/);
KVPOOL_API int kvpool_glt_find(kvpool_t* pool, uint64_t id, uint64_t* key, uint32_t* device_id, uint32_t* type, void** location,
                    kvpool_placement_t** pl, uint32_t* layer, uint32_t* block);
/* Whole-layer copies of the dense GLT columns (host[K_l] each; either may be NULL).                    */
KVPOOL_API int kvpool_layer_map(const kvpool_placement_t* pl, uint32_t layer, uint8_t* dev_out, uint32_t* slot_out);
KVPOOL_API const char* kvpool_last_error(void);
KVPOOL_API const char* kvpool_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KVPOOL_H */
