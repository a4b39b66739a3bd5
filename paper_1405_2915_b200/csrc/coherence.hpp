// The smart-container coherence protocol as a pure function (no CUDA): whole-container
// granularity, one host copy and one device copy (valid copies are reused,
// stale copies are never accessed, transfers are triggered only when the accessing unit has no valid
// copy; the protocol details are deferred by the paper to a thesis, so the table is DESIGN.md's
// "Coherence" reading).
#pragma once
#include <stddef.h>

namespace skel {

enum : int { ST_UNINIT = 0, ST_HOST = 1, ST_DEVICE = 2, ST_SHARED = 3 };  // bit0 host valid, bit1 device valid
enum : int { XFER_NONE = 0, XFER_H2D = 1, XFER_D2H = 2 };                 // bit mask
enum : int { ACTOR_DEVICE = 0, ACTOR_HOST = 1 };
enum : int { ACC_READ = 0, ACC_WRITE = 1, ACC_READWRITE = 2 };
enum : int { MODE_LAZY = 0, MODE_EAGER = 1 };

struct CoherenceStep {
  bool ok;        // false: the access would read a container that has no valid copy
  int new_state;  // state once the access (and, for a device access, the kernel) is done
  int transfer;   // XFER_H2D: before the kernel. XFER_D2H: host actor -> before the access;
                  // device actor (EAGER only) -> after the kernel.
};

inline CoherenceStep coherence_step(int state, int actor, int access, int mode) {
  const bool host_valid = state & 1, dev_valid = state & 2;
  const bool reads = access != ACC_WRITE, writes = access != ACC_READ;
  if (reads && state == ST_UNINIT) return {false, state, XFER_NONE};
  if (actor == ACTOR_HOST) {
    int xfer = XFER_NONE;
    if (reads && !host_valid) xfer = XFER_D2H;                 // only the device copy is valid
    const int ns = writes ? ST_HOST : (state | 1);             // a host write invalidates the device copy
    return {true, ns, xfer};
  }
  if (mode == MODE_LAZY) {
    int xfer = XFER_NONE;
    if (reads && !dev_valid) xfer = XFER_H2D;                  // upload only if the device has no valid copy
    const int ns = writes ? ST_DEVICE : (state | 2);           // WRITE of data about to be overwritten: no upload
    return {true, ns, xfer};
  }
  // EAGER baseline: upload every input that has a valid host copy, download every output, and
  // keep no device copy valid afterwards (a device-only container, e.g. an adopted buffer, is
  // used in place).
  int xfer = XFER_NONE;
  if (reads && host_valid) xfer |= XFER_H2D;
  int ns = host_valid ? ST_HOST : state;
  if (writes) {
    xfer |= XFER_D2H;
    ns = ST_HOST;
  }
  return {true, ns, xfer};
}

// ---- range extension ("partial copies ... when accessing a given range of elements") ----------
// A sorted list of disjoint, non-adjacent element ranges [begin, end): the parts of a container whose HOST copy is
// newer than the device copy (written through a host range access while the device copy stayed valid). Pure data
// structure, no CUDA: tested on the CPU through skel_ranges_add.
struct ElemRange { unsigned long long begin, end; };

// merge [begin, end) into the sorted disjoint list `r` of `count` ranges (capacity >= count + 1); returns the new count
inline size_t ranges_add(ElemRange* r, size_t count, unsigned long long begin, unsigned long long end) {
  if (begin >= end) return count;
  size_t i = 0;
  while (i < count && r[i].end < begin) ++i;          // ranges entirely before (not even adjacent)
  size_t j = i;
  while (j < count && r[j].begin <= end) {             // ranges that overlap or touch [begin, end)
    if (r[j].begin < begin) begin = r[j].begin;
    if (r[j].end > end) end = r[j].end;
    ++j;
  }
  if (j == i) {                                        // nothing to merge: insert at i
    for (size_t k = count; k > i; --k) r[k] = r[k - 1];
    r[i] = {begin, end};
    return count + 1;
  }
  r[i] = {begin, end};                                 // replace r[i..j) by the union
  for (size_t k = j; k < count; ++k) r[i + 1 + (k - j)] = r[k];
  return count - (j - i) + 1;
}

}  // namespace skel
