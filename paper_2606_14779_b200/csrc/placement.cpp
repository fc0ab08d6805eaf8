// Host-side placement arithmetic and stripe allocation.  See placement.hpp.
#include "placement.hpp"

#include <algorithm>
#include <cmath>
#include <numeric>

namespace kvp {

bool quantise_weights(const double* b, uint32_t n, uint64_t* w) {
  for (uint32_t i = 0; i < n; ++i) {
    if (!std::isfinite(b[i])) return false;
    const double mbps = std::floor(b[i] * 1000.0 + 0.5);
    if (mbps < 1.0 || mbps > 1.0e15) return false;
    w[i] = static_cast<uint64_t>(mbps);
  }
  return true;
}

void target_counts(const uint64_t* w, uint32_t n, uint64_t K, uint32_t* counts) {
  using u128 = unsigned __int128;
  u128 W = 0;
  for (uint32_t i = 0; i < n; ++i) W += w[i];
  uint64_t sum = 0;
  for (uint32_t i = 0; i < n; ++i) {
    counts[i] = static_cast<uint32_t>(static_cast<u128>(w[i]) * K / W);
    sum += counts[i];
  }
  // K - sum <= n-1 extras, one each, to the devices with the larger ratio (lower index on ties)
  uint32_t order[kMaxDevices];
  std::iota(order, order + n, 0u);
  std::stable_sort(order, order + n, [&](uint32_t a, uint32_t b) { return w[a] > w[b]; });
  for (uint64_t r = 0; r < K - sum; ++r) counts[order[r]] += 1;
}

void wrr_closed_form(const uint32_t* c, uint32_t n, uint64_t K, uint8_t* dev, uint32_t* slot) {
  (void)K;
  for (uint32_t i = 0; i < n; ++i) {
    const uint64_t ci = c[i];
    for (uint64_t k = 1; k <= ci; ++k) {
      uint64_t pos = k - 1;
      for (uint32_t o = 0; o < n; ++o) {
        if (o == i || c[o] == 0) continue;
        const uint64_t x = k * c[o];                 // < 2^64: k <= c_i < 2^32
        pos += (o < i) ? x / ci : (x - 1) / ci;     // floor(x/ci)  |  ceil(x/ci) - 1
      }
      dev[pos] = static_cast<uint8_t>(i);
      slot[pos] = static_cast<uint32_t>(k - 1);
    }
  }
}

StripeAllocator::StripeAllocator(uint64_t capacity, uint64_t align) : capacity_(capacity), align_(align) {
  if (capacity_ > 0) free_[0] = capacity_;
}

bool StripeAllocator::alloc(uint64_t size, uint64_t* offset_out) {
  if (size == 0) { *offset_out = 0; return true; }
  const uint64_t need = round_up(size);
  for (auto it = free_.begin(); it != free_.end(); ++it) {
    if (it->second < need) continue;
    const uint64_t off = it->first, len = it->second;
    free_.erase(it);
    if (len > need) free_[off + need] = len - need;
    used_ += need;
    *offset_out = off;
    return true;
  }
  return false;
}

void StripeAllocator::free(uint64_t offset, uint64_t size) {
  if (size == 0) return;
  uint64_t len = round_up(size);
  used_ -= len;
  auto next = free_.lower_bound(offset);
  if (next != free_.begin()) {
    auto prev = std::prev(next);
    if (prev->first + prev->second == offset) { offset = prev->first; len += prev->second; free_.erase(prev); }
  }
  if (next != free_.end() && offset + len == next->first) { len += next->second; free_.erase(next); }
  free_[offset] = len;
}

}  // namespace kvp
