// Host-side placement arithmetic and stripe allocation (a1-a4 of DESIGN.md §2).
// Pure C++17, no CUDA.  Cites: Eq. 1-2; Algorithm 1 l.4-16 PAPER.md:196-219.
#pragma once
#include <cstdint>
#include <map>
#include <vector>

namespace kvp {

constexpr uint32_t kMaxDevices = 32;

// Eq. 1.  w_i = floor(b_i*1000 + 0.5); false if any w_i < 1 or not finite.
bool quantise_weights(const double* bandwidth_gbps, uint32_t n, uint64_t* w_out);

// Eq. 2 + Alg. 1 l.8-12.  counts[i] = floor(w_i*K/W) (+1 for the first K - sum floors devices in
// (w desc, index asc) order).
void target_counts(const uint64_t* w, uint32_t n, uint64_t K, uint32_t* counts);

// Alg. 1 l.13-16 as smooth weighted round-robin, evaluated in closed form: the k-th block (1-based) of
// device i sits at enumeration position
//     (k-1) + sum_{i'<i} floor(k*c_i'/c_i) + sum_{i'>i} (ceil(k*c_i'/c_i) - 1)
// which is its rank when all (k/c_i, i) pairs are sorted — every (device, slot) is independent of the
// others, so there is no sequential loop over blocks.  dev/slot are indexed by logical block j.
void wrr_closed_form(const uint32_t* counts, uint32_t n, uint64_t K, uint8_t* dev, uint32_t* slot);

// First-fit free-list allocator over one pool buffer (byte offsets; coalesces on free).
class StripeAllocator {
 public:
  StripeAllocator() = default;
  explicit StripeAllocator(uint64_t capacity, uint64_t align = 4096);
  // Returns false if no range fits.  size 0 succeeds with offset 0 and reserves nothing.
  bool alloc(uint64_t size, uint64_t* offset_out);
  void free(uint64_t offset, uint64_t size);
  uint64_t used() const { return used_; }
  uint64_t capacity() const { return capacity_; }

 private:
  uint64_t round_up(uint64_t x) const { return (x + align_ - 1) / align_ * align_; }
  uint64_t capacity_ = 0, align_ = 4096, used_ = 0;
  std::map<uint64_t, uint64_t> free_;  // offset -> size
};

}  // namespace kvp
