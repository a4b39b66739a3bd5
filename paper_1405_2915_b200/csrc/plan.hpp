// Execution plans ("a run-time data structure ... for fast lookup of the expected
// best back-end ... and tunable parameters"; L53: "precomputing a tree-based dispatch structure for fast
// runtime lookup" from off-line sample executions). Pure host code, no CUDA.
//
// A tuned point is (instance key) -> sorted size breakpoints -> kernel variant. The keys form a DISPATCH TREE over the
// call context, one level per dimension, in this order:
//     skeleton -> dtype -> (fn, fn2) -> shape class / mode -> r0 -> r1 -> edge policy -> size breakpoints
// A lookup walks the tree from the root. Where the call's value has a child, it takes it; where it has not
// (a radius, edge policy, user function or shape class that was never tuned), it takes the NEAREST tuned child:
// for the radii the one closest in log2(r + 1), ties to the larger radius; for the categorical levels the first
// child. skeleton and dtype must match exactly. So r = 5, 6, 12 inherit the plan of r = 4, 8, 16, CYCLIC edges
// inherit DUPLICATE's, and only a (skeleton, dtype) pair with no tuned point at all falls back to the static
// preference list. The caller still checks that the inherited variant is applicable to the call.
#pragma once
#include <stddef.h>
#include <stdint.h>
#include <array>
#include <map>
#include <memory>
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
  // variant for n, or -1 if no tuned point shares the call's skeleton and dtype. *exact (optional) tells whether the
  // call's own key was tuned (true) or a neighbour's breakpoints were inherited (false). Binary search over the
  // breakpoints; below the first breakpoint -> the first entry's variant.
  int lookup(const InstanceKey& k, size_t n, bool* exact = nullptr) const;
  void set(const InstanceKey& k, size_t n_min, int variant);
  void erase(const InstanceKey& k);
  void clear();
  bool save(const char* path) const;
  bool load(const char* path);  // lines starting with '#' are comments (provenance)
  size_t size() const { return table_.size(); }
  // number of tree levels below the root (diagnostic)
  static constexpr int kLevels = 7;

 private:
  // level order of the tree: indices into InstanceKey::f, fn and fn2 merged into one level
  struct Node {
    std::map<int64_t, std::unique_ptr<Node>> child;
    const std::vector<Breakpoint>* leaf = nullptr;  // set on the last level
  };
  static int64_t level_value(const InstanceKey& k, int level);
  static bool level_is_radius(int level) { return level == 4 || level == 5; }
  void rebuild();
  std::map<InstanceKey, std::vector<Breakpoint>> table_;
  Node root_;
};

}  // namespace skel
