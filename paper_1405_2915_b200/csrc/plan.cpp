#include "plan.hpp"
#include <stdio.h>

namespace skel {

// text format, one instance per line:
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
  int version = 0;
  std::map<InstanceKey, std::vector<Breakpoint>> t;
  bool ok = fscanf(f, " skelplan %d", &version) == 1 && version == 1;
  while (ok) {
    InstanceKey k;
    int got = 0;
    for (int i = 0; i < 8; ++i) got += fscanf(f, "%d", &k.f[i]) == 1;
    if (got == 0) break;  // end of file
    size_t count = 0;
    if (got != 8 || fscanf(f, "%zu", &count) != 1 || count > 4096) { ok = false; break; }
    std::vector<Breakpoint> b(count);
    for (size_t i = 0; i < count && ok; ++i) {
      ok = fscanf(f, "%zu %d", &b[i].n_min, &b[i].variant) == 2;
      if (ok && i > 0 && b[i].n_min <= b[i - 1].n_min) ok = false;
    }
    if (ok) t[k] = b;
  }
  fclose(f);
  if (ok) table_.swap(t);
  return ok;
}

}  // namespace skel
