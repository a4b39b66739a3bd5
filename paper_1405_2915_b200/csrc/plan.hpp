// Execution plans ("a run-time data structure ... for fast lookup of the expected
// best back-end ... and tunable parameters"; L53: dispatch structures precomputed off-line from
// sample executions). Here: per skeleton instance, sorted size breakpoints -> kernel variant. Pure host
// code, no CUDA.
#pragma once
#include <stddef.h>
#include <stdint.h>
#include <array>
#include <map>
#include <string>
#include <vector>

namespace skel {

struct InstanceKey {
  std::array<int32_t, 8> f;  // skeleton, fn, fn2, dtype, r0, r1, edge, mode
  bool operator<(const InstanceKey& o) const { return f < o.f; }
};

struct Breakpoint { size_t n_min; int variant; };

class Plan {
 public:
  // variant for n, or -1 if the instance has no entry (binary search over the breakpoints;
  // below the first breakpoint -> the first entry's variant)
  int lookup(const InstanceKey& k, size_t n) const {
    auto it = table_.find(k);
    if (it == table_.end() || it->second.empty()) return -1;
    const std::vector<Breakpoint>& b = it->second;
    size_t lo = 0, hi = b.size();  // last entry with n_min <= n
    while (hi - lo > 1) {
      const size_t mid = (lo + hi) / 2;
      if (b[mid].n_min <= n) lo = mid; else hi = mid;
    }
    return b[lo].variant;
  }
  void set(const InstanceKey& k, size_t n_min, int variant) {
    std::vector<Breakpoint>& b = table_[k];
    size_t i = 0;
    while (i < b.size() && b[i].n_min < n_min) ++i;
    if (i < b.size() && b[i].n_min == n_min) b[i].variant = variant;
    else b.insert(b.begin() + i, Breakpoint{n_min, variant});
  }
  void erase(const InstanceKey& k) { table_.erase(k); }
  void clear() { table_.clear(); }
  bool save(const char* path) const;
  bool load(const char* path);
  size_t size() const { return table_.size(); }

 private:
  std::map<InstanceKey, std::vector<Breakpoint>> table_;
};

}  // namespace skel
