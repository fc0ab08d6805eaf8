/* A plain C99 client of include/kvpool.h: proves the header is valid C and that the boundary needs nothing but
 * pointers and sizes.  Uses only the pure-host entry points, so it runs without a GPU; with one argument "gpu" it
 * also creates a pool, places a request and prints the GLT entry of one block.  Built and run by tests/test_host_logic.py. */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "kvpool.h"

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
    if (argc > 1 && strcmp(argv[1], "gpu") == 0) {
        kvpool_device_desc d[2] = {{2.0, 8u << 20, -1, 0, -1, 0}, {1.0, 8u << 20, -1, KVPOOL_DEV_HBM, -1, 0}};
        kvpool_geometry g = {2, 16, 2, 64, 2};
        kvpool_t *pool = NULL;
        kvpool_placement_t *pl = NULL;
        uint32_t bpl[2] = {64, 3}, id, type, s;
        void *ptr;
        if (kvpool_create(d, 2, &g, 0, 0, &pool) != KVPOOL_OK) { fprintf(stderr, "%s\n", kvpool_last_error()); return 3; }
        if (kvpool_place(pool, bpl, &pl) != KVPOOL_OK) return 3;
        if (kvpool_lookup(pl, 0, 63, &id, &type, &s, &ptr) != KVPOOL_OK) return 3;
        printf("glt block 63: device %u type %u slot %u ptr %s\n", id, type, s, ptr ? "set" : "null");
        if (kvpool_lookup(pl, 0, 2, &id, &type, &s, &ptr) != KVPOOL_OK) return 3;
        printf("glt block 2: device %u type %u slot %u ptr %s\n", id, type, s, ptr ? "set" : "null");
        if (kvpool_release(pool, pl) != KVPOOL_OK || kvpool_destroy(pool) != KVPOOL_OK) return 3;
    }
    return 0;
}
