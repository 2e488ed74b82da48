// Scratch arena with lifetime-based reuse (BASELINE.json L5 item 6; "the full time frame must
// fit in GPU memory ... the reusage of memory for sequential steps of the tracking algorithm").
//
// Every scratch array of the tracker is declared with the first and last pipeline step that touches it.  The
// planner places each array at the lowest offset of ONE caller-provided device buffer that does not collide
// with an already placed array whose lifetime overlaps (largest arrays first).  Arrays of sequential steps
// therefore share addresses (e.g. the selector's claim array reuses the sort rank + raw link region), and
// the plan is fixed at create time: no allocation, no synchronisation at tracking time.
#pragma once
#include <algorithm>
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

namespace tpc {

struct ArenaAlloc {
  std::string name;
  size_t bytes = 0;
  int first_step = 0, last_step = 0;
  size_t offset = 0;
};

class ArenaPlan {
 public:
  static constexpr size_t kAlign = 256;

  // returns the id of the allocation
  int add(const char* name, size_t bytes, int first_step, int last_step) {
    ArenaAlloc a;
    a.name = name;
    a.bytes = (bytes + kAlign - 1) / kAlign * kAlign;
    a.first_step = first_step;
    a.last_step = last_step;
    allocs_.push_back(a);
    return (int)allocs_.size() - 1;
  }

  void plan() {
    std::vector<int> order(allocs_.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return allocs_[a].bytes > allocs_[b].bytes; });
    std::vector<int> placed;
    peak_ = 0;
    for (int id : order) {
      ArenaAlloc& a = allocs_[id];
      // candidate offsets: 0 and the end of every conflicting placed allocation
      std::vector<size_t> cands{0};
      for (int p : placed) if (overlaps_in_time(a, allocs_[p])) cands.push_back(allocs_[p].offset + allocs_[p].bytes);
      std::sort(cands.begin(), cands.end());
      for (size_t off : cands) {
        bool ok = true;
        for (int p : placed) {
          const ArenaAlloc& b = allocs_[p];
          if (overlaps_in_time(a, b) && off < b.offset + b.bytes && b.offset < off + a.bytes) { ok = false; break; }
        }
        if (ok) { a.offset = off; break; }
      }
      placed.push_back(id);
      peak_ = std::max(peak_, a.offset + a.bytes);
    }
  }

  size_t peak_bytes() const { return peak_; }
  size_t sum_bytes() const { size_t s = 0; for (const auto& a : allocs_) s += a.bytes; return s; }
  const std::vector<ArenaAlloc>& allocs() const { return allocs_; }
  template <typename T> T* ptr(void* base, int id) const { return reinterpret_cast<T*>(static_cast<char*>(base) + allocs_[id].offset); }

 private:
  static bool overlaps_in_time(const ArenaAlloc& a, const ArenaAlloc& b) {
    return a.first_step <= b.last_step && b.first_step <= a.last_step;
  }
  std::vector<ArenaAlloc> allocs_;
  size_t peak_ = 0;
};

}  // namespace tpc
