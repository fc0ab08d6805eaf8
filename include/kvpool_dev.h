/*
 * kvpool_dev.h — development entry points of libkvpool.so: comparison baselines, consumer stand-ins, work counters and
 * per-kernel profiling.  bench.py and the tests use them to produce the evidence DESIGN.md quotes; an engine that moves
 * KV needs only kvpool.h.  Same library, same conventions (kvpool.h header comment): every call returns KVPOOL_OK or a
 * negative KVPOOL_E* code, "host" / "device" says where a pointer's memory lives, nothing here is a product path and
 * nothing here is part of the paper's method (the operations the paper defines are all in kvpool.h).
 */
#ifndef KVPOOL_DEV_H
#define KVPOOL_DEV_H

#include "kvpool.h"

#ifdef __cplusplus
extern "C" {
#endif

/* kvpool_set_profiling modes */
#define KVPOOL_PROFILE_OFF 0
#define KVPOOL_PROFILE_SIDE 1
#define KVPOOL_PROFILE_INSTREAM 2


/* Comparison baseline, not a product path: what an engine without a gather kernel does — one cudaMemcpyAsync per
 * K block and per V block (2*K_l calls) straight between the paged blocks and the stripes, all on `stream`.
 * block_table_host is the HOST copy of the layer's table.  Same results as kvpool_offload / kvpool_retrieve;
 * exists so that bench.py --variants can time it next to the kernel paths.                                        */
KVPOOL_API int kvpool_offload_naive(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, const void* k_base /*device*/,
                         const void* v_base /*device*/, uint64_t block_stride_bytes, const int32_t* block_table_host, void* cuda_stream);
KVPOOL_API int kvpool_retrieve_naive(kvpool_t* pool, kvpool_placement_t* pl, uint32_t layer, void* k_base /*device*/, void* v_base /*device*/,
                          uint64_t block_stride_bytes, const int32_t* block_table_host, void* cuda_stream);

/* Consumer stand-in and integrity check (the "GPU computation" box of Fig. 2, for pipeline
 * experiments; not part of the paper's method).  Adds to *sum_dev (device uint64, caller zeroes it) the checksum
 *     sum over logical blocks j < n_blocks, halves h (0 = K, 1 = V), 64-bit little-endian words i of
 *         word(j, h, i) * (2*idx + 1)   mod 2^64,      idx = (j*2 + h)*(kvb/8) + i
 * of the paged blocks named by block_table_dev, reading them through the table as decode attention would
 * (n_blocks*P bytes of HBM reads).  kvb must be a multiple of 16.  Ordered on `stream`.                          */
KVPOOL_API int kvpool_checksum(kvpool_t* pool, const void* k_base /*device*/, const void* v_base /*device*/, uint64_t block_stride_bytes,
                    const int32_t* block_table_dev, uint32_t n_blocks, uint64_t* sum_dev /*device*/, void* cuda_stream);
/* The consumer side of kvpool_retrieve_layers_signal in one host call (what a serving engine's C++ layer loop does; a Python
 * loop of 2 x n_layers calls costs more host time than a 1K-token request takes to arrive): for q = 0 .. n_layers-1,
 * `stream` waits for layer_ready[q] (cudaEvent_t; NULL = no wait) and then runs kvpool_checksum over layer q's
 * n_blocks[q] blocks into sums_dev[q].  k_bases / v_bases / block_tables_dev / layer_ready / n_blocks are HOST arrays of
 * n_layers entries; sums_dev is a device array of n_layers uint64 the caller has zeroed.                            */
KVPOOL_API int kvpool_checksum_layers(kvpool_t* pool, uint32_t n_layers, const void* const* k_bases /*host[n] of device*/,
                           const void* const* v_bases, uint64_t block_stride_bytes, const int32_t* const* block_tables_dev,
                           const uint32_t* n_blocks /*host[n]*/, void* const* layer_ready /*host[n] of cudaEvent_t, or NULL*/,
                           uint64_t* sums_dev /*device[n]*/, void* cuda_stream);
/* Occupy `stream` for `nanoseconds` with a one-thread kernel (calibrated compute stand-in).                        */
KVPOOL_API int kvpool_spin(kvpool_t* pool, uint64_t nanoseconds, void* cuda_stream);


/* Work counters since create: kernels launched and cudaMemcpyAsync calls issued by the library.        */
KVPOOL_API int kvpool_stats(const kvpool_t* pool, uint64_t* kernel_launches, uint64_t* memcpy_calls);

/* Per-kernel timing for the roofline report.  While enabled, every kernel the library launches is bracketed by a
 * CUDA timing-event pair taken after all of the launch's stream waits (so a pair spans the kernel alone, not the
 * transfers it waited for).  enabled = KVPOOL_PROFILE_SIDE (1): the launching stream only gets two non-timing marker
 * events and the timing events are recorded on two side streams of the pool behind those markers — a TIMING event
 * recorded on the launching stream itself holds that stream up until its timestamp is written (3 us on an idle GPU,
 * 25-47 us under a concurrent copy-engine transfer over the host link), which both delays the kernel and counts the
 * delay.  KVPOOL_PROFILE_INSTREAM (2) records the pair on the launching stream anyway, for comparison.  kvpool_profile_read blocks until the recorded pairs of `kind`
 * have completed, returns their summed duration, count and algorithmic bytes (K_l*P per launch), and clears them.
 * kind: 0 = in-device pack, 1 = in-device unpack, 2 = zero-copy offload, 3 = zero-copy retrieve.               */
KVPOOL_API int kvpool_set_profiling(kvpool_t* pool, int enabled);
KVPOOL_API int kvpool_profile_read(kvpool_t* pool, int kind, double* total_ms, uint64_t* launches, uint64_t* bytes);
/* The same read plus the kernels' own clock: while profiling is on, every CTA of a launch folds its start and its end
 * (%globaltimer, after its stores are globally visible) into a per-launch {min start, max end} pair in device memory;
 * device_ms is the sum of (max end - min start) over the device_launches launches that got such a pair (the first
 * 16384 between two reads that empty the record list).  The event pairs of total_ms also count what the stream's front
 * end adds around a launch — ~5 us on an idle GPU, 20-35 us while a copy engine streams over the host link (an empty
 * event pair measures the same) — device_ms does not.  Any out pointer may be NULL.                   */
KVPOOL_API int kvpool_profile_read_clock(kvpool_t* pool, int kind, double* total_ms, double* device_ms, uint64_t* launches,
                              uint64_t* device_launches, uint64_t* bytes);


#ifdef __cplusplus
}
#endif
#endif /* KVPOOL_DEV_H */
