/* A plain C99 client of include/kvpool.h: proves the header is valid C and that the boundary needs nothing but
 * pointers and sizes.  Without arguments it uses only the pure-host entry points, so it runs without a GPU (built and
 * run by tests/test_host_logic.py).  With the argument "gpu" (tests/test_gpu_parity.py) it also moves bytes: it creates
 * a pool of one pinned host device and one HBM-type device, places a request, offloads a small paged layer it filled
 * itself, retrieves it into a poisoned copy and compares — the round trip, the untouched blocks, and one payload on
 * each pool device located through kvpool_lookup (Table I `location`).  With a file name as second argument the pool gets
 * a third, SSD-type device backed by that file (KV-passthrough): its payloads are found by LBA
 * (kvpool_ssd_location) and read back with plain pread.  It links the library and the CUDA runtime only: no oracle, no
 * Python. */
#define _XOPEN_SOURCE 700
#include <fcntl.h>
#include <unistd.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "kvpool.h"


/* the five CUDA runtime calls the client needs, declared here so that the file stays plain C99 without CUDA headers */
extern int cudaMalloc(void **p, size_t n);
extern int cudaFree(void *p);
extern int cudaMemcpy(void *dst, const void *src, size_t n, int kind); /* 1 = host->device, 2 = device->host */
extern int cudaMemset(void *p, int v, size_t n);
extern int cudaDeviceSynchronize(void);

#define CHECK(x) do { if ((x) != 0) { fprintf(stderr, "%s failed: %s\n", #x, kvpool_last_error()); return 3; } } while (0)

static int gpu_round_trip(const char *ssd_path) {
    enum { NPHYS = 96, K0 = 64, K1 = 3, KVB = 16 * 2 * 64 * 2, PLANE = NPHYS * KVB };
    kvpool_device_desc d[3] = {{2.0, 8u << 20, -1, 0, -1, 0, NULL, 0, 0}, {1.0, 8u << 20, -1, KVPOOL_DEV_HBM, -1, 0, NULL, 0, 0},
                               {1.0, 8u << 20, -1, KVPOOL_DEV_SSD, -1, 0, NULL, 512, 0}};
    const uint32_t n_dev = ssd_path ? 3 : 2;
    uint64_t lba = 0;
    uint32_t in_sector = 0, sector = 0;
    int fd = -1;
    kvpool_geometry g = {2, 16, 2, 64, 2};
    kvpool_t *pool = NULL;
    kvpool_placement_t *pl = NULL;
    uint32_t bpl[2] = {K0, K1}, id, type, s, x = 14779u, seen[3] = {0, 0, 0};
    int32_t table[K0];
    unsigned char *src = malloc(2 * PLANE), *back = malloc(2 * PLANE), *payload = malloc(2 * KVB);
    void *src_d = NULL, *dst_d = NULL, *table_d = NULL, *ptr = NULL;
    size_t i;
    int j;
    if (!src || !back || !payload) return 3;
    for (i = 0; i < 2 * (size_t)PLANE; ++i) { x = x * 1664525u + 1013904223u; src[i] = (unsigned char)(x >> 24); }
    for (j = 0; j < K0; ++j) table[j] = (j * 37 + 11) % NPHYS; /* 37 is coprime with 96: distinct physical blocks */
    CHECK(kvpool_validate_table(table, K0, NPHYS));
    d[2].path = ssd_path;
    CHECK(kvpool_create(d, n_dev, &g, 0, 0, &pool));
    CHECK(kvpool_place(pool, bpl, &pl));
    CHECK(kvpool_lookup(pl, 0, 63, &id, &type, &s, &ptr));
    printf("glt block 63: device %u type %u slot %u ptr %s\n", id, type, s, ptr ? "set" : "null");
    CHECK(kvpool_lookup(pl, 0, 2, &id, &type, &s, &ptr));
    printf("glt block 2: device %u type %u slot %u ptr %s\n", id, type, s, ptr ? "set" : "null");
    CHECK(cudaMalloc(&src_d, 2 * PLANE));
    CHECK(cudaMalloc(&dst_d, 2 * PLANE));
    CHECK(cudaMalloc(&table_d, sizeof table));
    CHECK(cudaMemcpy(src_d, src, 2 * PLANE, 1));
    CHECK(cudaMemcpy(table_d, table, sizeof table, 1));
    CHECK(cudaMemset(dst_d, 0xC1, 2 * PLANE));
    CHECK(cudaDeviceSynchronize());
    /* Alg. 1 l.17-22: store; then wait until the stripes are complete in the pool */
    CHECK(kvpool_offload(pool, pl, 0, src_d, (char *)src_d + PLANE, KVB, table_d, NULL));
    CHECK(kvpool_wait_offloads(pool, pl, NULL));
    CHECK(cudaDeviceSynchronize());
    CHECK(kvpool_synchronize(pool));
    /* Table I: every block's payload (K block then V block) sits at its `location` */
    for (j = 0; j < K0; ++j) {
        CHECK(kvpool_lookup(pl, 0, (uint32_t)j, &id, &type, &s, &ptr));
        if (id >= n_dev || type != (id == 2 ? (uint32_t)KVPOOL_TYPE_SSD : id ? (uint32_t)KVPOOL_TYPE_HBM : (uint32_t)KVPOOL_TYPE_MEM)) return 4;
        if (type == KVPOOL_TYPE_MEM) memcpy(payload, ptr, 2 * KVB);
        else if (type == KVPOOL_TYPE_HBM) CHECK(cudaMemcpy(payload, ptr, 2 * KVB, 2));
        else { /* Table I: type SSD, location = LBA; SSD_Direct_Retrieve by hand */
            CHECK(kvpool_ssd_location(pl, 0, (uint32_t)j, &lba, &in_sector));
            CHECK(kvpool_ssd_range(pl, 0, id, NULL, NULL, &sector));
            if ((uint64_t)(size_t)ptr != lba) return 4;
            if (fd < 0 && (fd = open(ssd_path, O_RDONLY)) < 0) return 4;
            if (pread(fd, payload, 2 * KVB, (off_t)(lba * sector + in_sector)) != 2 * KVB) return 4;
        }
        if (memcmp(payload, src + (size_t)table[j] * KVB, KVB) || memcmp(payload + KVB, src + PLANE + (size_t)table[j] * KVB, KVB)) {
            fprintf(stderr, "payload of block %d differs from the paged K/V block\n", j);
            return 4;
        }
        seen[id]++;
    }
    printf("payloads ok: %u on the host device, %u on the HBM device\n", seen[0], seen[1]);
    if (ssd_path) printf("payloads ok: %u on the SSD device (%u-byte sectors)\n", seen[2], sector);
    if (fd >= 0) close(fd);
    /* retrieve into the poisoned copy */
    CHECK(kvpool_retrieve(pool, pl, 0, dst_d, (char *)dst_d + PLANE, KVB, table_d, NULL));
    CHECK(cudaDeviceSynchronize());
    CHECK(cudaMemcpy(back, dst_d, 2 * PLANE, 2));
    for (j = 0; j < K0; ++j) { /* the request's blocks are back, bit for bit; mark them as checked */
        size_t o = (size_t)table[j] * KVB;
        if (memcmp(back + o, src + o, KVB) || memcmp(back + PLANE + o, src + PLANE + o, KVB)) return 5;
        memset(back + o, 0xC1, KVB);
        memset(back + PLANE + o, 0xC1, KVB);
    }
    for (i = 0; i < 2 * (size_t)PLANE; ++i)
        if (back[i] != 0xC1) { fprintf(stderr, "byte %lu outside the request's blocks was written\n", (unsigned long)i); return 5; }
    printf("round trip ok: %d blocks of %d bytes, %d other blocks untouched\n", K0, 2 * KVB, NPHYS - K0);
    CHECK(kvpool_release(pool, pl));
    CHECK(kvpool_destroy(pool));
    cudaFree(src_d); cudaFree(dst_d); cudaFree(table_d);
    free(src); free(back); free(payload);
    return 0;
}

int main(int argc, char **argv) {
    const double bw[6] = {4.0, 4.0, 2.0, 2.0, 1.0, 1.0};
    uint64_t w[6];
    uint32_t counts[6], slot[64];
    uint8_t dev[64];
    if (kvpool_plan_weights(bw, 6, w) != KVPOOL_OK) { fprintf(stderr, "%s\n", kvpool_last_error()); return 1; }
    if (kvpool_plan_layer(w, 6, 8192, counts, NULL, NULL) != KVPOOL_OK) return 1;
    printf("counts %u %u %u %u %u %u\n", counts[0], counts[1], counts[2], counts[3], counts[4], counts[5]);
    if (kvpool_plan_layer(w, 6, 64, counts, dev, slot) != KVPOOL_OK) return 1;
    printf("dev");
    for (int j = 0; j < 16; ++j) printf(" %u", dev[j]);
    printf("\n");
    if (kvpool_plan_weights(bw, 0, w) != KVPOOL_EINVAL) return 2;
    printf("error \"%s\"\n", kvpool_last_error());
    printf("%s\n", kvpool_version());
    printf("sizeof %u %u %u\n", (unsigned)sizeof(kvpool_device_desc), (unsigned)sizeof(kvpool_geometry), (unsigned)sizeof(kvpool_tuning));
    if (argc > 1 && strcmp(argv[1], "gpu") == 0) return gpu_round_trip(argc > 2 ? argv[2] : NULL);
    return 0;
}
