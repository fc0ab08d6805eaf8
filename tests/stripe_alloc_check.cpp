// CPU check of the stripe allocator (a4) against a page-bitmap model: random alloc / free sequences;
// every returned range is aligned, inside the buffer, disjoint from every live range and the LOWEST gap that fits
// (first fit); used() equals the model's; after everything is freed the whole capacity is one range again (coalescing).
// Built and run by tests/test_host_logic.py with g++ (placement.cpp is plain C++17, no CUDA).
#include <cstdint>
#include <cstdio>
#include <random>
#include <vector>

#include "../paper_2606_14779_b200/csrc/placement.hpp"

using kvp::StripeAllocator;

struct Live { uint64_t off, size; };

static int fail(const char* what, uint64_t a, uint64_t b) {
  std::printf("FAIL %s (%llu, %llu)\n", what, (unsigned long long)a, (unsigned long long)b);
  return 1;
}

int main() {
  for (uint64_t align : {256ull, 4096ull}) {
    for (uint32_t seed = 0; seed < 20; ++seed) {
      std::mt19937_64 rng(14779 + seed);
      const uint64_t pages = 64 + rng() % 448, capacity = pages * align + (seed % 3 ? 0 : rng() % align);  // ragged capacity too
      StripeAllocator a(capacity, align);
      std::vector<char> busy(pages + 1, 0);
      std::vector<Live> live;
      uint64_t used = 0;
      for (int step = 0; step < 4000; ++step) {
        if (live.empty() || rng() % 100 < 55) {
          const uint64_t size = 1 + rng() % (align * (1 + rng() % 40));
          const uint64_t need = (size + align - 1) / align;
          // model: lowest run of `need` free pages that lies inside the capacity
          uint64_t want = ~0ull;
          for (uint64_t p = 0, run = 0; p < pages + 1; ++p) {
            const bool free_page = !busy[p] && (p + 1) * align <= capacity;
            run = free_page ? run + 1 : 0;
            if (run == need) { want = (p + 1 - need) * align; break; }
          }
          uint64_t off = 12345;
          const bool ok = a.alloc(size, &off);
          if (ok != (want != ~0ull)) return fail("alloc success differs from the model", size, want);
          if (!ok) continue;
          if (off != want) return fail("not the lowest fitting gap", off, want);
          if (off % align || off + need * align > capacity) return fail("misaligned or outside the buffer", off, size);
          for (uint64_t p = off / align; p < off / align + need; ++p) {
            if (busy[p]) return fail("overlaps a live range", off, p);
            busy[p] = 1;
          }
          used += need * align;
          live.push_back({off, size});
        } else {
          const size_t k = rng() % live.size();
          a.free(live[k].off, live[k].size);
          const uint64_t need = (live[k].size + align - 1) / align;
          for (uint64_t p = live[k].off / align; p < live[k].off / align + need; ++p) busy[p] = 0;
          used -= need * align;
          live[k] = live.back();
          live.pop_back();
        }
        if (a.used() != used) return fail("used() differs from the model", a.used(), used);
      }
      for (const Live& l : live) a.free(l.off, l.size);
      uint64_t off = 1;
      if (a.used() != 0) return fail("used() after freeing everything", a.used(), 0);
      if (!a.alloc(capacity / align * align, &off) || off != 0) return fail("free ranges did not coalesce", off, capacity);
      uint64_t z = 7;
      if (!a.alloc(0, &z) || z != 0) return fail("size 0", z, 0);
    }
  }
  std::printf("stripe allocator ok\n");
  return 0;
}
