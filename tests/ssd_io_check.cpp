// CPU-only driver for csrc/ssd_io.cpp (the host side of KV-passthrough): plays the GPU's half of every
// command with plain memcpy and the same two sequence flags, so that the worker thread, its read-modify-write of edge
// sectors, the zero padding of a range's last sector and the lane hand-over are exercised without a GPU.  The expected
// bytes are NOT computed here: tests/test_host_logic.py compares the backing file and the read-back with the oracle.
//
//   ssd_io_check <file> <sector> <kv_size> <first_lba> <lane_bytes> <n_lanes> <stripe.bin> <out.bin> <lo:hi> [<lo:hi> ...]
//
// stripe.bin holds the offload set's payloads in slot order; every <lo:hi> stores slots [lo, hi) of it (in the order given,
// in lane-sized commands); afterwards the whole set is retrieved through the lanes into out.bin.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../paper_2606_14779_b200/csrc/ssd_io.hpp"

using namespace kvp;

static std::vector<uint8_t> slurp(const char* path) {
  FILE* f = fopen(path, "rb");
  if (!f) { perror(path); exit(2); }
  std::vector<uint8_t> v;
  uint8_t buf[65536];
  size_t n;
  while ((n = fread(buf, 1, sizeof buf, f)) > 0) v.insert(v.end(), buf, buf + n);
  fclose(f);
  return v;
}

int main(int argc, char** argv) {
  if (argc < 10) { fprintf(stderr, "usage: see the header of this file\n"); return 2; }
  const char* file = argv[1];
  const uint32_t sector = static_cast<uint32_t>(atoi(argv[2]));
  const uint64_t P = strtoull(argv[3], nullptr, 10), first_lba = strtoull(argv[4], nullptr, 10), lane_bytes = strtoull(argv[5], nullptr, 10);
  const uint32_t lanes = static_cast<uint32_t>(atoi(argv[6]));
  const std::vector<uint8_t> stripe = slurp(argv[7]);
  const uint64_t slots = stripe.size() / P;
  SsdDevice dev;
  std::string err;
  uint64_t n_sec = 0;
  if (!lba_range_len(slots, P, sector, &n_sec)) return 3;
  int rc = dev.open(file, (first_lba + n_sec + 4) * sector, sector, &err);
  if (rc) { fprintf(stderr, "open: %s\n", err.c_str()); return 3; }
  const uint32_t stride = 32;
  uint8_t* bounce = static_cast<uint8_t*>(aligned_alloc(4096, 2ull * lanes * lane_bytes));
  uint32_t* flags = static_cast<uint32_t*>(aligned_alloc(4096, 2ull * lanes * stride * 4));
  memset(flags, 0, 2ull * lanes * stride * 4);
  uint8_t* const b2[2] = {bounce, bounce + lanes * lane_bytes};
  volatile uint32_t* const gpu[2] = {flags, flags + lanes * stride};
  volatile uint32_t* const cpu[2] = {flags + 16, flags + lanes * stride + 16};
  dev.start(lanes, lane_bytes, b2, gpu, cpu, stride);
  std::vector<uint32_t> use[2] = {std::vector<uint32_t>(lanes, 0), std::vector<uint32_t>(lanes, 0)};
  uint32_t cursor[2] = {0, 0};
  const uint64_t base = first_lba * sector;

  // one command over slots [x, x+n): the same arithmetic the library's chunker feeds the worker (byte offset -> sector + head)
  auto command = [&](bool store, uint64_t x, uint64_t n, uint8_t* out) {
    const int d = store ? 1 : 0;
    const uint64_t byte0 = base + x * P, at = byte0 / sector * sector;
    const uint32_t head = static_cast<uint32_t>(byte0 - at), k = cursor[d]++ % lanes, u = ++use[d][k];
    uint8_t* lane = b2[d] + k * lane_bytes;
    if (store) {
      while (!seq_reached(cpu[d] + k * stride, u - 1)) {}            // "cuStreamWaitValue32": the lane's previous store is on the disk
      memcpy(lane + head, stripe.data() + x * P, n * P);             // "the D2H copy"
      dev.submit(SsdCmd{SsdCmd::kWrite, x + n == slots, k, u, at, head, n * P});
      __atomic_store_n(gpu[d] + k * stride, u, __ATOMIC_RELEASE);    // "cuStreamWriteValue32"
    } else {
      dev.submit(SsdCmd{SsdCmd::kRead, false, k, u, at, head, n * P});
      while (!seq_reached(cpu[d] + k * stride, u)) {}
      memcpy(out + x * P, lane + head, n * P);                       // "the H2D copy"
      __atomic_store_n(gpu[d] + k * stride, u, __ATOMIC_RELEASE);
    }
  };
  auto span = [&](bool store, uint64_t lo, uint64_t hi, uint8_t* out) {
    for (uint64_t x = lo; x < hi;) {
      const uint64_t head = (base + x * P) % sector;
      uint64_t n = (lane_bytes - sector - head) / P;
      if (n == 0) { fprintf(stderr, "lane too small\n"); exit(3); }
      if (n > hi - x) n = hi - x;
      command(store, x, n, out);
      x += n;
    }
  };
  for (int a = 9; a < argc; ++a) {
    unsigned long long lo = 0, hi = 0;
    if (sscanf(argv[a], "%llu:%llu", &lo, &hi) != 2 || lo > hi || hi > slots) return 2;
    span(true, lo, hi, nullptr);
  }
  dev.drain();
  if (int e = dev.take_error()) { fprintf(stderr, "store failed: %s\n", strerror(e)); return 4; }
  std::vector<uint8_t> back(stripe.size(), 0xEE);
  span(false, 0, slots, back.data());
  dev.drain();
  if (int e = dev.take_error()) { fprintf(stderr, "retrieve failed: %s\n", strerror(e)); return 4; }
  FILE* f = fopen(argv[8], "wb");
  if (!f || fwrite(back.data(), 1, back.size(), f) != back.size()) return 5;
  fclose(f);
  printf("ssd io ok: %llu stores, %llu retrieves, direct=%d\n", (unsigned long long)dev.completed(1), (unsigned long long)dev.completed(0), dev.direct() ? 1 : 0);
  dev.close();
  free(bounce);
  free(flags);
  return 0;
}
