#include "plan.hpp"
#include <math.h>
#include <stdio.h>
#include <string.h>

namespace skel {

// tree levels: 0 skeleton, 1 dtype, 2 (fn, fn2), 3 mode / shape class, 4 r0, 5 r1, 6 edge
int64_t Plan::level_value(const InstanceKey& k, int level) {
  switch (level) {
    case 0: return k.f[0];
    case 1: return k.f[3];
    case 2: return (int64_t(k.f[1]) << 32) | uint32_t(k.f[2]);
    case 3: return k.f[7];
    case 4: return k.f[4];
    case 5: return k.f[5];
    default: return k.f[6];
  }
}

void Plan::rebuild() {
  root_.child.clear();
  for (const auto& kv : table_) {
    if (kv.second.empty()) continue;
    Node* n = &root_;
    for (int level = 0; level < kLevels; ++level) {
      std::unique_ptr<Node>& c = n->child[level_value(kv.first, level)];
      if (!c) c.reset(new Node);
      n = c.get();
    }
    n->leaf = &kv.second;  // std::map nodes are stable
  }
}

int Plan::lookup(const InstanceKey& k, size_t n, bool* exact) const {
  const Node* node = &root_;
  bool ex = true;
  for (int level = 0; level < kLevels; ++level) {
    const int64_t want = level_value(k, level);
    auto it = node->child.find(want);
    if (it == node->child.end()) {
      if (level < 2 || node->child.empty()) {  // skeleton and dtype must match
        if (exact) *exact = false;
        return -1;
      }
      ex = false;
      if (level_is_radius(level)) {  // nearest in log2(r + 1); ties -> the larger radius
        double best = 1e300;
        auto bestit = node->child.end();
        for (auto c = node->child.begin(); c != node->child.end(); ++c) {
          const double d = fabs(log2(double(c->first) + 1.0) - log2(double(want) + 1.0));
          if (bestit == node->child.end() || d < best - 1e-12 || (fabs(d - best) <= 1e-12 && c->first > bestit->first)) {
            best = d;
            bestit = c;
          }
        }
        it = bestit;
      } else {
        it = node->child.begin();
      }
    }
    node = it->second.get();
  }
  if (exact) *exact = ex;
  if (!node->leaf || node->leaf->empty()) return -1;
  const std::vector<Breakpoint>& b = *node->leaf;
  size_t lo = 0, hi = b.size();  // last entry with n_min <= n
  while (hi - lo > 1) {
    const size_t mid = (lo + hi) / 2;
    if (b[mid].n_min <= n) lo = mid; else hi = mid;
  }
  return b[lo].variant;
}

void Plan::set(const InstanceKey& k, size_t n_min, int variant) {
  const bool fresh = table_.find(k) == table_.end();
  std::vector<Breakpoint>& b = table_[k];
  size_t i = 0;
  while (i < b.size() && b[i].n_min < n_min) ++i;
  if (i < b.size() && b[i].n_min == n_min) b[i].variant = variant;
  else b.insert(b.begin() + i, Breakpoint{n_min, variant});
  if (fresh) rebuild();
}

void Plan::erase(const InstanceKey& k) {
  if (table_.erase(k)) rebuild();
}

void Plan::clear() {
  table_.clear();
  rebuild();
}

// text format, one tuned point per line ('#' starts a comment line):
//   skelplan 1
//   <skeleton> <fn> <fn2> <dtype> <r0> <r1> <edge> <mode> <count> (<n_min> <variant>)*count
bool Plan::save(const char* path) const {
  FILE* f = fopen(path, "w");
  if (!f) return false;
  fprintf(f, "skelplan 1\n");
  for (const auto& kv : table_) {
    for (int i = 0; i < 8; ++i) fprintf(f, "%d ", kv.first.f[i]);
    fprintf(f, "%zu", kv.second.size());
    for (const Breakpoint& b : kv.second) fprintf(f, " %zu %d", b.n_min, b.variant);
    fprintf(f, "\n");
  }
  return fclose(f) == 0;
}

bool Plan::load(const char* path) {
  FILE* f = fopen(path, "r");
  if (!f) return false;
  std::map<InstanceKey, std::vector<Breakpoint>> t;
  bool ok = true, header = false;
  char line[65536];
  while (ok && fgets(line, sizeof line, f)) {
    char* p = line;
    while (*p == ' ' || *p == '\t') ++p;
    if (*p == '#' || *p == '\n' || *p == '\r' || *p == 0) continue;
    if (!header) {
      int version = 0;
      ok = sscanf(p, "skelplan %d", &version) == 1 && version == 1;
      header = true;
      continue;
    }
    InstanceKey k;
    int used = 0, pos = 0;
    for (int i = 0; i < 8 && ok; ++i) {
      ok = sscanf(p + pos, "%d%n", &k.f[i], &used) == 1;
      pos += used;
    }
    size_t count = 0;
    ok = ok && sscanf(p + pos, "%zu%n", &count, &used) == 1 && count >= 1 && count <= 4096;
    pos += used;
    std::vector<Breakpoint> b(ok ? count : 0);
    for (size_t i = 0; i < b.size() && ok; ++i) {
      ok = sscanf(p + pos, "%zu %d%n", &b[i].n_min, &b[i].variant, &used) == 2;
      pos += used;
      if (ok && i > 0 && b[i].n_min <= b[i - 1].n_min) ok = false;
    }
    if (ok) t[k] = b;
  }
  fclose(f);
  ok = ok && header;
  if (ok) {
    table_.swap(t);
    rebuild();
  }
  return ok;
}

}  // namespace skel
