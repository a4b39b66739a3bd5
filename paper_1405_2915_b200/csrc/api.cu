// C ABI of libskel.so (include/skel.h): contexts, smart containers with the coherence protocol,
// skeleton entry points, variant selection and tuning. Host code only; kernels live in the other
// translation units (kernels.hpp).
#include "../../include/skel.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <limits>
#include <new>
#include <string>
#include <vector>

#include "coherence.hpp"
#include "kernels.hpp"
#include "plan.hpp"
#include <memory>
#include <time.h>

using namespace skel;

namespace {

constexpr uint32_t MAGIC_CTX = 0x534b4358, MAGIC_VEC = 0x534b5645, MAGIC_MAT = 0x534b4d41, MAGIC_FUT = 0x534b4655;
constexpr int FUTURE_SLOTS = 1024;  // outstanding skel_future per context (8-byte pinned slots)
constexpr int FN_IDENT_ = 100;  // same value as skel::FN_IDENT in common.cuh (identity map of plain Reduce)

struct Storage {
  skel_ctx* ctx;
  int dtype;
  size_t n;
  void* host = nullptr;  // pinned, library owned, allocated on first host use
  void* dev = nullptr;
  bool dev_owned = true;
  int state = ST_UNINIT;
  bool host_held = false;
  int refs = 1;
  // data-dependence tracking: ctx->seq of the last enqueued stream operation that touched the
  // container in any way / that wrote one of its copies. A host READ waits for the last writer only, a host WRITE
  // for both; the wait is on the event recorded after THAT operation (EventRing), never on the whole stream.
  uint64_t last_seq = 0;
  uint64_t last_write_seq = 0;
  // range-granular coherence: element ranges whose HOST copy is newer than the (otherwise valid) device copy.
  // Non-empty only while the device-valid bit of `state` is set.
  std::vector<ElemRange> host_newer;
  // skel_*_prefetch_host: a download in flight on the context's copy stream (nullptr = none). The host copy counts
  // as valid in `state`; host accesses and device writes wait for this event first.
  cudaEvent_t d2h_done = nullptr;
};

struct Handle {
  uint32_t magic;
  Storage* st;
  size_t rows, cols;  // vectors: rows = 1, cols = n
};

}  // namespace

// One event per enqueued operation, kept in a ring: slot i holds an event recorded on the context's stream when every
// operation with sequence number <= seq[i] had been enqueued. To wait for operation q, synchronise on the recorded slot
// with the smallest seq >= q (the stream is in order: a later event implies the earlier operations). A slot that has
// been reused only makes the wait conservative, never wrong.
struct EventRing {
  static constexpr int N = 64;
  cudaEvent_t ev[N] = {};
  uint64_t seq[N] = {};
  int head = 0;
};

struct PendingCall;
struct RecordedCall;
struct skel_future {
  uint32_t magic;
  skel_ctx* ctx;
  int slot;      // index of its pinned scalar slot
  int dtype;
  uint64_t seq;  // sequence number of the reducing operation
};
struct skel_vector : Handle {};
struct skel_matrix : Handle {};

struct skel_ctx {
  uint32_t magic = MAGIC_CTX;
  cudaStream_t stream = nullptr;
  skel_alloc_fn alloc = nullptr;
  skel_free_fn free_ = nullptr;
  void* user = nullptr;
  int mode = MODE_LAZY;
  skel_stats stats{};
  std::string err;
  int live = 0;
  bool dev_ready = false;
  int sms = 148;
  Scratch scratch{};
  unsigned* tile_ctr = nullptr;  // device: tile counter of the persistent TMA kernels (kernels.hpp Launch)
  unsigned tile_next = 0;        // host: its value when the next launch starts
  void* d_result = nullptr;  // device slot for scalars returned to the host
  void* h_result = nullptr;      // pinned, mapped host slot for scalars returned to the host ...
  void* h_result_dev = nullptr;  // ... and its device-side address: the reducing kernel stores the scalar straight into it
  uint64_t seq = 0;           // sequence number of the last stream operation issued (launch or copy)
  uint64_t done_seq = 0;      // every operation <= done_seq is known to have finished
  uint64_t recorded_seq = 0;  // every operation <= recorded_seq is covered by an event of the ring
  EventRing ring;
  // skel_*_async: pinned, mapped scalar slots the reducing kernels write their result into (zero-copy)
  void* h_slots = nullptr;
  void* h_slots_dev = nullptr;
  std::vector<int> free_slots;
  bool sticky = false;
  Plan plan;
  int forced[SKEL_SK_COUNT];
  int last_sk = -1, last_var = -1;
  int launches = 0;
  std::vector<float> tune_table;
  // L2-aware traversal direction of Reduce / MapReduce (launch_now)
  bool l2_reuse = true, reverse_next = false, walk_reverse = false;
  const void* walk_in0 = nullptr;   // first operand of the last launch_now launch
  uint64_t walk_launch = ~0ull;     // kernels launched by the context up to and including it
  // cross-call fusion (skel_ctx_set_fusion): launches of a fusible chain are held back here
  bool fusion = false;
  std::vector<struct PendingCall> pending;
  // skel_replay_*: the calls recorded between _begin and _end (call, operands, variant)
  bool recording = false;
  std::vector<struct RecordedCall> recorded;
  cudaStream_t copy_stream = nullptr;  // skel_*_prefetch_host: downloads that overlap the compute stream's work
  void* sep_tmp = nullptr;  // intermediate matrix of the two-pass separable MapOverlap
  size_t sep_tmp_bytes = 0;
  void* spare = nullptr;  // buffer an in-place Map of a fused chain writes into (then swapped with the container's)
  size_t spare_bytes = 0;
};

namespace {

skel_status fail(skel_ctx* c, skel_status s, const char* msg) {
  if (c) c->err = msg;
  return s;
}

skel_status cuda_fail(skel_ctx* c, cudaError_t e, const char* where) {
  c->sticky = true;
  c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return SKEL_ERR_CUDA;
}

#define CU(ctx, call)                                      \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

bool ctx_ok(const skel_ctx* c) { return c && c->magic == MAGIC_CTX; }
bool vec_ok(const skel_vector* v) { return v && v->magic == MAGIC_VEC && v->st; }
bool mat_ok(const skel_matrix* m) { return m && m->magic == MAGIC_MAT && m->st; }

size_t esize(int dtype) { return dtype == SKEL_F64 ? 8 : 4; }

skel_status ensure_device(skel_ctx* c) {
  if (c->sticky) return SKEL_ERR_CUDA;
  if (c->dev_ready) return SKEL_OK;
  int dev = 0;
  CU(c, cudaGetDevice(&dev));
  CU(c, cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev));
  char* base = nullptr;
  const size_t partial_bytes = size_t(MAX_PARTIALS) * 8;
  CU(c, cudaMalloc(reinterpret_cast<void**>(&base), 2 * partial_bytes + 512));
  CU(c, cudaMemsetAsync(base, 0, 2 * partial_bytes + 512, c->stream));
  c->scratch.red_tagged = reinterpret_cast<unsigned long long*>(base + partial_bytes + 256);
  c->scratch.red_epoch = 0;
  c->scratch.partials = base;
  c->scratch.ticket = reinterpret_cast<unsigned*>(base + partial_bytes);
  c->scratch.scan_ticket = reinterpret_cast<unsigned*>(base + partial_bytes + 64);
  c->d_result = base + partial_bytes + 128;
  c->tile_ctr = reinterpret_cast<unsigned*>(base + partial_bytes + 192);
  c->tile_next = 0;
  c->scratch.scan_state = nullptr;
  c->scratch.scan_state_tiles = 0;
  c->scratch.scan_epoch = 0;
  CU(c, cudaHostAlloc(&c->h_result, 64, cudaHostAllocMapped));
  CU(c, cudaHostGetDevicePointer(&c->h_result_dev, c->h_result, 0));
  c->dev_ready = true;
  return SKEL_OK;
}

skel_status ensure_scan_state(skel_ctx* c, size_t n) {
  const size_t need = scan_tiles_needed(n);
  if (need <= c->scratch.scan_state_tiles) return SKEL_OK;
  if (c->scratch.scan_state) {
    CU(c, cudaStreamSynchronize(c->stream));
    CU(c, cudaFree(c->scratch.scan_state));
    c->scratch.scan_state = nullptr;
    c->scratch.scan_state_tiles = 0;
  }
  size_t cap = 1024;
  while (cap < need) cap *= 2;
  CU(c, cudaMalloc(reinterpret_cast<void**>(&c->scratch.scan_state), cap * 8));
  CU(c, cudaMemsetAsync(c->scratch.scan_state, 0, cap * 8, c->stream));
  c->scratch.scan_state_tiles = cap;
  c->scratch.scan_epoch = 0;
  return SKEL_OK;
}

// fp64 single-pass scan: 16 bytes of state per 4096-element tile (f64.cu). The array is zero-filled once and never
// cleared: states are tagged with a launch number that never repeats. Growing it waits for the stream (rare).
skel_status ensure_scan_state64(skel_ctx* c, size_t n) {
  const size_t need = scan_f64_state_words(n);
  if (need <= c->scratch.scan_state64_words) return SKEL_OK;
  if (c->scratch.scan_state64) {
    CU(c, cudaStreamSynchronize(c->stream));
    CU(c, cudaFree(c->scratch.scan_state64));
    c->scratch.scan_state64 = nullptr;
    c->scratch.scan_state64_words = 0;
  }
  size_t cap = 2048;
  while (cap < need) cap *= 2;
  CU(c, cudaMalloc(reinterpret_cast<void**>(&c->scratch.scan_state64), cap * 8));
  CU(c, cudaMemsetAsync(c->scratch.scan_state64, 0, cap * 8, c->stream));
  c->scratch.scan_state64_words = cap;
  return SKEL_OK;
}

skel_status dev_alloc(skel_ctx* c, size_t bytes, void** out) {
  *out = nullptr;
  if (bytes == 0) return SKEL_OK;
  if (c->alloc) {
    *out = c->alloc(bytes, c->stream, c->user);
    if (!*out) return fail(c, SKEL_ERR_OOM, "device allocator callback returned NULL");
    return SKEL_OK;
  }
  cudaError_t e = cudaMalloc(out, bytes);
  if (e == cudaErrorMemoryAllocation) {
    cudaGetLastError();
    return fail(c, SKEL_ERR_OOM, "cudaMalloc: out of memory");
  }
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc");
  return SKEL_OK;
}

void dev_free(skel_ctx* c, void* p) {
  if (!p) return;
  if (c->alloc) {
    if (c->free_) c->free_(p, c->user);
  } else {
    cudaFree(p);
  }
}

skel_status ensure_host(skel_ctx* c, Storage* s) {
  if (s->host || s->n == 0) return SKEL_OK;
  cudaError_t e = cudaHostAlloc(&s->host, s->n * esize(s->dtype), cudaHostAllocDefault);
  if (e == cudaErrorMemoryAllocation) {
    cudaGetLastError();
    return fail(c, SKEL_ERR_OOM, "cudaHostAlloc: out of memory");
  }
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaHostAlloc");
  return SKEL_OK;
}

skel_status flush_pending(skel_ctx* c);
bool has_pending(const skel_ctx* c);
skel_status mark_enqueued(skel_ctx* c);

// a prefetch download in flight: block the host until it has landed
skel_status finish_prefetch(skel_ctx* c, Storage* s) {
  if (!s->d2h_done) return SKEL_OK;
  cudaError_t e = cudaEventSynchronize(s->d2h_done);
  cudaEventDestroy(s->d2h_done);
  s->d2h_done = nullptr;
  if (e != cudaSuccess) return cuda_fail(c, e, "prefetch download");
  return SKEL_OK;
}

// ... or make the compute stream wait for it (before a kernel overwrites the device buffer it reads from)
skel_status order_after_prefetch(skel_ctx* c, Storage* s) {
  if (!s->d2h_done) return SKEL_OK;
  CU(c, cudaStreamWaitEvent(c->stream, s->d2h_done, 0));
  return SKEL_OK;
}

// upload the ranges the host has written since the device copy was last made current (device copy stays valid)
skel_status upload_host_newer(skel_ctx* c, Storage* s) {
  if (s->host_newer.empty()) return SKEL_OK;
  skel_status st = flush_pending(c);  // keep the stream order
  if (st != SKEL_OK) return st;
  const size_t es = esize(s->dtype);
  for (const ElemRange& r : s->host_newer) {
    const size_t bytes = size_t(r.end - r.begin) * es;
    CU(c, cudaMemcpyAsync(static_cast<char*>(s->dev) + r.begin * es, static_cast<char*>(s->host) + r.begin * es, bytes,
                          cudaMemcpyHostToDevice, c->stream));
    c->stats.h2d_bytes += bytes;
    c->stats.h2d_count += 1;
  }
  s->host_newer.clear();
  s->last_seq = ++c->seq;
  return SKEL_OK;
}

void add_host_newer(Storage* s, size_t begin, size_t end) {
  s->host_newer.resize(s->host_newer.size() + 1);
  const size_t cnt = ranges_add(s->host_newer.data(), s->host_newer.size() - 1, begin, end);
  s->host_newer.resize(cnt);
}

// Every operation issued so far has been enqueued on the stream (nothing is held back): cover them with an event.
skel_status mark_enqueued(skel_ctx* c) {
  if (c->recorded_seq == c->seq || has_pending(c)) return SKEL_OK;
  EventRing& r = c->ring;
  if (!r.ev[r.head]) CU(c, cudaEventCreateWithFlags(&r.ev[r.head], cudaEventDisableTiming));
  CU(c, cudaEventRecord(r.ev[r.head], c->stream));
  r.seq[r.head] = c->seq;
  c->recorded_seq = c->seq;
  r.head = (r.head + 1) % EventRing::N;
  return SKEL_OK;
}

// the recorded event that covers operation q (the one with the smallest seq >= q), or nullptr when q is known to have
// finished; operations not yet covered by an event are launched / covered first
skel_status event_for(skel_ctx* c, uint64_t q, cudaEvent_t* ev, uint64_t* ev_seq) {
  *ev = nullptr;
  *ev_seq = 0;
  if (q <= c->done_seq) return SKEL_OK;
  if (q > c->recorded_seq) {
    skel_status st = flush_pending(c);
    if (st != SKEL_OK) return st;
    st = mark_enqueued(c);
    if (st != SKEL_OK) return st;
  }
  const EventRing& r = c->ring;
  int best = -1;
  for (int i = 0; i < EventRing::N; ++i)
    if (r.ev[i] && r.seq[i] >= q && (best < 0 || r.seq[i] < r.seq[best])) best = i;
  if (best < 0) return fail(c, SKEL_ERR_CUDA, "internal: no event covers a pending operation");
  *ev = r.ev[best];
  *ev_seq = r.seq[best];
  return SKEL_OK;
}

// block the host until operation `q` (and, the stream being in order, everything before it) has finished
skel_status wait_seq(skel_ctx* c, uint64_t q) {
  cudaEvent_t ev;
  uint64_t ev_seq;
  skel_status st = event_for(c, q, &ev, &ev_seq);
  if (st != SKEL_OK || !ev) return st;
  CU(c, cudaEventSynchronize(ev));
  if (ev_seq > c->done_seq) c->done_seq = ev_seq;
  return SKEL_OK;
}

// Download elements [offset, offset + count) of `s` to its host copy on the context's COPY stream, ordered after the
// last operation that wrote the container (its event), not after everything enqueued on the compute stream: a host
// read of a container whose producer has finished does not wait for unrelated kernels enqueued since. s->d2h_done
// fires when the data has landed; until then a device write to the container waits for it (order_after_prefetch).
skel_status start_download(skel_ctx* c, Storage* s, size_t offset, size_t count) {
  if (!c->copy_stream) CU(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
  cudaEvent_t produced;
  uint64_t produced_seq;
  skel_status st = event_for(c, s->last_write_seq, &produced, &produced_seq);
  if (st != SKEL_OK) return st;
  if (produced) CU(c, cudaStreamWaitEvent(c->copy_stream, produced, 0));
  const size_t es = esize(s->dtype);
  CU(c, cudaMemcpyAsync(static_cast<char*>(s->host) + offset * es, static_cast<char*>(s->dev) + offset * es, count * es,
                        cudaMemcpyDeviceToHost, c->copy_stream));
  if (!s->d2h_done) CU(c, cudaEventCreateWithFlags(&s->d2h_done, cudaEventDisableTiming));
  CU(c, cudaEventRecord(s->d2h_done, c->copy_stream));
  c->stats.d2h_bytes += count * es;
  c->stats.d2h_count += 1;
  return SKEL_OK;
}

// host access to `s`: a read waits for the last operation that wrote one of its copies, a write for the last one
// that touched it at all (a device read of the buffer the host is about to overwrite included)
skel_status wait_for(skel_ctx* c, Storage* s, bool host_writes = true) {
  return wait_seq(c, host_writes ? s->last_seq : s->last_write_seq);
}

// ---- containers --------------------------------------------------------------------------------
template <typename H>
skel_status make_handle(skel_ctx* c, uint32_t magic, int dt, size_t rows, size_t cols, H** out) {
  if (!ctx_ok(c) || !out) return fail(ctx_ok(c) ? c : nullptr, SKEL_ERR_INVALID_ARG, "NULL context or out pointer");
  *out = nullptr;
  if (dt != SKEL_F32 && dt != SKEL_I32 && dt != SKEL_F64) return fail(c, SKEL_ERR_INVALID_ARG, "unknown dtype");
  if (cols != 0 && rows > std::numeric_limits<size_t>::max() / 8 / cols)
    return fail(c, SKEL_ERR_INVALID_ARG, "size overflow");
  Storage* s = new (std::nothrow) Storage;
  H* h = new (std::nothrow) H;
  if (!s || !h) {
    delete s;
    delete h;
    return fail(c, SKEL_ERR_OOM, "host allocation failed");
  }
  s->ctx = c;
  s->dtype = dt;
  s->n = rows * cols;
  h->magic = magic;
  h->st = s;
  h->rows = rows;
  h->cols = cols;
  ++c->live;
  *out = h;
  return SKEL_OK;
}

skel_status flush_pending(skel_ctx* c);

skel_status release_handle(Handle* h) {
  Storage* s = h->st;
  skel_ctx* c = s->ctx;
  if (s->host_held && s->refs == 1) return fail(c, SKEL_ERR_BUSY, "host access is still held");
  flush_pending(c);  // a held-back launch may still reference this container
  if (s->refs == 1) finish_prefetch(c, s);
  if (--s->refs == 0) {
    if (!c->sticky) wait_seq(c, s->last_seq);
    if (s->dev_owned) dev_free(c, s->dev);
    if (s->host) cudaFreeHost(s->host);
    delete s;
  }
  h->magic = 0;
  h->st = nullptr;
  --c->live;
  return SKEL_OK;
}

skel_status fill_from(skel_ctx* c, Storage* s, const void* src) {
  if (s->n == 0) {
    s->state = ST_HOST;
    return SKEL_OK;
  }
  if (!src) return fail(c, SKEL_ERR_INVALID_ARG, "src is NULL");
  skel_status st = ensure_device(c);  // pinned allocations need the CUDA context
  if (st != SKEL_OK) return st;
  st = ensure_host(c, s);
  if (st != SKEL_OK) return st;
  memcpy(s->host, src, s->n * esize(s->dtype));
  s->state = ST_HOST;
  return SKEL_OK;
}

skel_status host_acquire(Handle* h, skel_access mode, void** host_ptr) {
  Storage* s = h->st;
  skel_ctx* c = s->ctx;
  if (!host_ptr) return fail(c, SKEL_ERR_INVALID_ARG, "host_ptr is NULL");
  if (mode != SKEL_READ && mode != SKEL_WRITE && mode != SKEL_READWRITE)
    return fail(c, SKEL_ERR_INVALID_ARG, "bad access mode");
  if (s->host_held) return fail(c, SKEL_ERR_BUSY, "host access already held");
  {
    skel_status pst = finish_prefetch(c, s);
    if (pst != SKEL_OK) return pst;
  }
  const CoherenceStep step = coherence_step(s->state, ACTOR_HOST, mode, c->mode);
  if (!step.ok) return fail(c, SKEL_ERR_UNINIT, "host read of a container that was never written");
  skel_status st = flush_pending(c);
  if (st != SKEL_OK) return st;
  if (!s->host_newer.empty()) {
    // ranges written through a host range access: a whole-container read of a host copy that is otherwise invalid
    // must not lose them (make the device current first, then download); an access that leaves the host copy the
    // only valid one makes the list moot; a read of a fully valid host copy keeps it.
    if (step.transfer & XFER_D2H) {
      st = upload_host_newer(c, s);
      if (st != SKEL_OK) return st;
    } else if (!(step.new_state & 2)) {
      s->host_newer.clear();
    }
  }
  if (s->n > 0) {
    st = ensure_device(c);
    if (st != SKEL_OK) return st;
    st = ensure_host(c, s);
    if (st != SKEL_OK) return st;
    if (step.transfer & XFER_D2H) {
      st = start_download(c, s, 0, s->n);
      if (st != SKEL_OK) return st;
      st = finish_prefetch(c, s);
      if (st != SKEL_OK) return st;
    }
    st = wait_for(c, s, mode != SKEL_READ);
    if (st != SKEL_OK) return st;
  }
  s->state = step.new_state;
  s->host_held = true;
  *host_ptr = s->host;
  return SKEL_OK;
}

skel_status host_release(Handle* h) {
  Storage* s = h->st;
  if (!s->host_held) return fail(s->ctx, SKEL_ERR_INVALID_ARG, "host access is not held");
  s->host_held = false;
  return SKEL_OK;
}

// Asynchronous download on the copy stream (include/skel.h skel_vector_prefetch_host).
skel_status prefetch_host(Handle* h) {
  Storage* s = h->st;
  skel_ctx* c = s->ctx;
  if (s->host_held) return fail(c, SKEL_ERR_BUSY, "container is held by the host");
  if (s->state != ST_DEVICE || s->n == 0) return SKEL_OK;  // nothing to do: the host copy is (becoming) valid
  skel_status st = finish_prefetch(c, s);  // an earlier download whose result a device write has made stale since
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = ensure_host(c, s);
  if (st != SKEL_OK) return st;
  st = upload_host_newer(c, s);  // ranges the host wrote must not be overwritten by the download
  if (st != SKEL_OK) return st;
  st = start_download(c, s, 0, s->n);  // ordered after the container's last writer (the producing kernel)
  if (st != SKEL_OK) return st;
  s->state = ST_SHARED;  // valid once d2h_done has fired: every host access waits for it
  return SKEL_OK;
}

// Range-granular host access (include/skel.h skel_vector_host_acquire_range).
skel_status host_acquire_range(Handle* h, skel_access mode, size_t offset, size_t count, void** host_ptr) {
  Storage* s = h->st;
  skel_ctx* c = s->ctx;
  if (!host_ptr) return fail(c, SKEL_ERR_INVALID_ARG, "host_ptr is NULL");
  if (mode != SKEL_READ && mode != SKEL_WRITE && mode != SKEL_READWRITE) return fail(c, SKEL_ERR_INVALID_ARG, "bad access mode");
  if (count == 0 || offset > s->n || count > s->n - offset) return fail(c, SKEL_ERR_INVALID_ARG, "range out of bounds");
  if (s->host_held) return fail(c, SKEL_ERR_BUSY, "host access already held");
  if (s->state == ST_UNINIT) return fail(c, SKEL_ERR_UNINIT, "range access to a container that was never written");
  skel_status st = finish_prefetch(c, s);
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = ensure_host(c, s);
  if (st != SKEL_OK) return st;
  const size_t es = esize(s->dtype);
  const bool host_valid = s->state & 1, dev_valid = s->state & 2;
  if (!host_valid && mode != SKEL_WRITE) {
    // only this range comes down; parts of it the host has written since are newer than the device's: make the
    // device current first if they overlap
    for (const ElemRange& r : s->host_newer)
      if (r.begin < offset + count && offset < r.end) {
        st = upload_host_newer(c, s);
        if (st != SKEL_OK) return st;
        break;
      }
    st = start_download(c, s, offset, count);
    if (st != SKEL_OK) return st;
    st = finish_prefetch(c, s);
    if (st != SKEL_OK) return st;
  }
  st = wait_for(c, s, mode != SKEL_READ);  // a host write also waits for device reads of the host buffer still in flight
  if (st != SKEL_OK) return st;
  if (mode != SKEL_READ && dev_valid) add_host_newer(s, offset, offset + count);
  s->host_held = true;
  *host_ptr = static_cast<char*>(s->host) + offset * es;
  return SKEL_OK;
}

// ---- operand acquisition for a skeleton call -----------------------------------------------------
struct Operand {
  Storage* st;
  int access;
  CoherenceStep step;
};

struct OperandSet {
  Operand ops[4];
  int count = 0;
  void add(Storage* s, int access) {
    for (int i = 0; i < count; ++i)
      if (ops[i].st == s) {
        if (ops[i].access != access) ops[i].access = ACC_READWRITE;
        return;
      }
    ops[count++] = Operand{s, access, {}};
  }
};

void record_call(skel_ctx* c, const OperandSet& set);  // skel_replay_*: defined next to run_call

skel_status acquire_all(skel_ctx* c, OperandSet& set) {
  skel_status st = ensure_device(c);
  if (st != SKEL_OK) return st;
  for (int i = 0; i < set.count; ++i) {  // validate everything before any side effect
    Operand& o = set.ops[i];
    if (o.st->ctx != c) return fail(c, SKEL_ERR_INVALID_ARG, "container belongs to another context");
    if (o.st->host_held) return fail(c, SKEL_ERR_BUSY, "container is held by the host");
    o.step = coherence_step(o.st->state, ACTOR_DEVICE, o.access, c->mode);
    if (!o.step.ok) return fail(c, SKEL_ERR_UNINIT, "skeleton input was never written");
  }
  // Two DIFFERENT containers of a call must not share device memory when one of them is written (possible only with
  // skel_*_adopt_device over overlapping buffers): the kernels choose non-coherent loads, halo reads and in-place
  // forms by container identity, so such a call would race silently. One handle used as input and output is fine.
  for (int i = 0; i < set.count; ++i)
    for (int j = i + 1; j < set.count; ++j) {
      const Storage* a = set.ops[i].st;
      const Storage* b = set.ops[j].st;
      if (!a->dev || !b->dev || a->n == 0 || b->n == 0) continue;
      if (set.ops[i].access == ACC_READ && set.ops[j].access == ACC_READ) continue;
      const char* a0 = static_cast<const char*>(a->dev);
      const char* b0 = static_cast<const char*>(b->dev);
      if (a0 < b0 + b->n * esize(b->dtype) && b0 < a0 + a->n * esize(a->dtype))
        return fail(c, SKEL_ERR_ALIAS, "two containers of this call overlap in device memory (adopted buffers)");
    }
  for (int i = 0; i < set.count; ++i) {
    Operand& o = set.ops[i];
    Storage* s = o.st;
    if (!s->dev && s->n > 0) {
      st = dev_alloc(c, s->n * esize(s->dtype), &s->dev);
      if (st != SKEL_OK) return st;
    }
    if (s->d2h_done && (o.access != ACC_READ || (o.step.transfer & XFER_H2D))) {
      st = order_after_prefetch(c, s);  // the download still reads the device buffer this call overwrites
      if (st != SKEL_OK) return st;
    }
    if (!s->host_newer.empty()) {
      if (o.access == ACC_WRITE || (o.step.transfer & XFER_H2D)) s->host_newer.clear();  // overwritten / uploaded whole
      else {
        st = upload_host_newer(c, s);  // the device copy is valid except for these ranges
        if (st != SKEL_OK) return st;
      }
    }
    if ((o.step.transfer & XFER_H2D) && s->n > 0) {
      st = flush_pending(c);  // keep the stream order: held-back launches go first
      if (st != SKEL_OK) return st;
      CU(c, cudaMemcpyAsync(s->dev, s->host, s->n * esize(s->dtype), cudaMemcpyHostToDevice, c->stream));
      c->stats.h2d_bytes += s->n * esize(s->dtype);
      c->stats.h2d_count += 1;
    } else if (o.access != ACC_WRITE && !(o.step.transfer & XFER_H2D)) {
      c->stats.h2d_elided += 1;
    }
  }
  return SKEL_OK;
}

skel_status publish_all(skel_ctx* c, OperandSet& set) {
  const uint64_t seq = ++c->seq;
  for (int i = 0; i < set.count; ++i) {
    Operand& o = set.ops[i];
    Storage* s = o.st;
    if (o.step.transfer & XFER_D2H) {  // EAGER: download the output right after the kernel
      if (s->n > 0) {
        skel_status st = flush_pending(c);
        if (st != SKEL_OK) return st;
        st = ensure_host(c, s);
        if (st != SKEL_OK) return st;
        CU(c, cudaMemcpyAsync(s->host, s->dev, s->n * esize(s->dtype), cudaMemcpyDeviceToHost, c->stream));
        c->stats.d2h_bytes += s->n * esize(s->dtype);
        c->stats.d2h_count += 1;
      }
    } else if (o.access != ACC_READ) {
      c->stats.d2h_elided += 1;
    }
    s->state = o.step.new_state;
    s->last_seq = seq;
    if (o.access != ACC_READ || (o.step.transfer & (XFER_H2D | XFER_D2H))) s->last_write_seq = seq;
  }
  c->stats.launches += c->launches;
  c->launches = 0;
  if (c->recording) record_call(c, set);
  return mark_enqueued(c);  // no-op while the launch is held back (fusion): flush_pending records it
}

// ---- calls, variants ---------------------------------------------------------------------------
struct Call {
  skel_instance inst{};
  const void* in0 = nullptr;
  const void* in1 = nullptr;
  const void* in2 = nullptr;  // three-vector Map
  void* out = nullptr;
  size_t n = 0, rows = 1, cols = 0;
  uint32_t cbits = 0;  // constant c / scan init, as the element type's bits (32-bit element types)
  float pad = 0.f;
  // fp64 elements (f64.cu): constant / scan init / pad as doubles, weights behind a pointer (the struct stays small)
  double c64 = 0.0, pad64 = 0.0;
  std::shared_ptr<const Weights1D64> w1_64;
  std::shared_ptr<const Weights2D64> w2_64;
  Weights1D w1;
  Weights2D w2;
  Weights1D w1b;  // separable: the column filter (w1 = the row filter, r0 / r1 = their radii)
  Storage* in_st = nullptr;   // containers behind in0 / out (fusion: buffer swap of an in-place Map)
  Storage* out_st = nullptr;
};
}  // namespace
struct PendingCall { Call k; };
struct RecordedCall { Call k; OperandSet set; int variant; };
namespace {

InstanceKey key_of(const skel_instance& i) {
  InstanceKey k;
  k.f = {i.skeleton, i.fn, i.fn2, i.dtype, i.r0, i.r1, i.edge, i.mode};
  return k;
}

int variant_count(int sk) {
  switch (sk) {
    case SKEL_SK_MAP: return map_variant_count();
    case SKEL_SK_REDUCE:
    case SKEL_SK_MAPREDUCE: return reduce_variant_count();
    case SKEL_SK_SCAN: return scan_variant_count();
    case SKEL_SK_OVERLAP1D: return overlap1d_variant_count();
    case SKEL_SK_OVERLAP1D_COL: return overlap1d_col_variant_count();
    case SKEL_SK_OVERLAP2D: return overlap2d_variant_count();
    case SKEL_SK_SEPARABLE: return separable_variant_count();
    case SKEL_SK_REDUCE_ROWS: return reduce_rows_variant_count();
  }
  return 0;
}

const char* variant_name(int sk, int v) {
  switch (sk) {
    case SKEL_SK_MAP: return map_variant_name(v);
    case SKEL_SK_REDUCE:
    case SKEL_SK_MAPREDUCE: return reduce_variant_name(v);
    case SKEL_SK_SCAN: return scan_variant_name(v);
    case SKEL_SK_OVERLAP1D: return overlap1d_variant_name(v);
    case SKEL_SK_OVERLAP1D_COL: return overlap1d_col_variant_name(v);
    case SKEL_SK_OVERLAP2D: return overlap2d_variant_name(v);
    case SKEL_SK_SEPARABLE: return separable_variant_name(v);
    case SKEL_SK_REDUCE_ROWS: return reduce_rows_variant_name(v);
  }
  return nullptr;
}

bool variant_ok(const Call& k, int v) {
  switch (k.inst.skeleton) {
    case SKEL_SK_MAP:
      return map_variant_ok(v, k.in0, k.in1, k.out, k.n) && (k.in2 == nullptr || map_variant_ok(v, k.in2, nullptr, k.out, k.n));
    case SKEL_SK_REDUCE:
    case SKEL_SK_MAPREDUCE: return reduce_variant_ok(v, k.in0, k.in1, k.n);
    case SKEL_SK_SCAN: return scan_variant_ok(v, k.inst.dtype, k.in0, k.out, k.n);
    case SKEL_SK_OVERLAP1D: return overlap1d_variant_ok(v, k.inst.dtype, k.inst.r0, k.in0, k.out, k.rows, k.cols);
    case SKEL_SK_OVERLAP1D_COL: return overlap1d_col_variant_ok(v, k.inst.dtype, k.inst.r0, k.in0, k.out, k.rows, k.cols);
    case SKEL_SK_OVERLAP2D: return overlap2d_variant_ok(v, k.inst.dtype, k.inst.r0, k.inst.r1, k.in0, k.out, k.rows, k.cols);
    case SKEL_SK_SEPARABLE: return separable_variant_ok(v, k.inst.r0, k.inst.r1, k.in0, k.out, k.rows, k.cols);
    case SKEL_SK_REDUCE_ROWS: return reduce_rows_variant_ok(v, k.in0, k.rows, k.cols);
  }
  return false;
}

// Untuned defaults: preference order per skeleton; the last entry runs every call.
const int* preference(int sk, int dtype, int* count) {
  static const int map_p[] = {2, 1, 0};
  static const int red_p[] = {1, 0};
  static const int scan_i[] = {15, 3, 0, 4, 5};
  static const int scan_f[] = {4, 5};
  static const int o1_p[] = {2, 1, 0};
  static const int o1_i[] = {10, 8, 4, 0};  // int32 elements: tma_swz_o16_s3, regshfl_2x8, regshfl_o16, direct
  static const int tma_i[] = {5, 0};        // int32 columns / 2D: tma_oy4, direct
  static const int col_p[] = {2, 0};
  static const int o2_p[] = {1, 0};
  static const int sep_p[] = {4, 1, 0};
  static const int rows_p[] = {1, 0};
  switch (sk) {
    case SKEL_SK_MAP: *count = 3; return map_p;
    case SKEL_SK_REDUCE:
    case SKEL_SK_MAPREDUCE: *count = 2; return red_p;
    case SKEL_SK_SCAN:
      if (dtype == SKEL_I32) { *count = 5; return scan_i; }
      *count = 2; return scan_f;
    case SKEL_SK_OVERLAP1D:
      if (dtype == SKEL_I32) { *count = 4; return o1_i; }
      *count = 3; return o1_p;
    case SKEL_SK_OVERLAP1D_COL:
      if (dtype == SKEL_I32) { *count = 2; return tma_i; }
      *count = 2; return col_p;
    case SKEL_SK_OVERLAP2D:
      if (dtype == SKEL_I32) { *count = 2; return tma_i; }
      *count = 2; return o2_p;
    case SKEL_SK_SEPARABLE: *count = 3; return sep_p;
    case SKEL_SK_REDUCE_ROWS: *count = 2; return rows_p;
  }
  *count = 0;
  return nullptr;
}

skel_status choose_variant(skel_ctx* c, const Call& k, int* chosen) {
  const int sk = k.inst.skeleton;
  const int forced = c->forced[sk];
  if (forced >= 0) {
    if (forced >= variant_count(sk) || !variant_ok(k, forced))
      return fail(c, SKEL_ERR_UNSUPPORTED, "forced variant is not applicable to this call");
    *chosen = forced;
    return SKEL_OK;
  }
  int v = c->plan.lookup(key_of(k.inst), k.n);
  if (v >= 0 && v < variant_count(sk) && variant_ok(k, v)) {
    *chosen = v;
    return SKEL_OK;
  }
  int cnt = 0;
  const int* pref = preference(sk, k.inst.dtype, &cnt);
  for (int i = 0; i < cnt; ++i)
    if (variant_ok(k, pref[i])) {
      *chosen = pref[i];
      return SKEL_OK;
    }
  return fail(c, SKEL_ERR_UNSUPPORTED, "no applicable kernel variant");
}

cudaError_t launch_call(skel_ctx* c, const Call& k, int v);

// the two 1D passes through the context's temporary matrix, each with the variant its own plan picks
cudaError_t launch_separable_two_pass(skel_ctx* c, const Call& k) {
  const size_t bytes = k.rows * k.cols * sizeof(float);
  if (c->sep_tmp_bytes < bytes) {
    if (c->sep_tmp) dev_free(c, c->sep_tmp);
    c->sep_tmp = nullptr;
    c->sep_tmp_bytes = 0;
    if (dev_alloc(c, bytes, &c->sep_tmp) != SKEL_OK) return cudaErrorMemoryAllocation;
    c->sep_tmp_bytes = bytes;
  }
  Call p = k;
  p.inst.skeleton = SKEL_SK_OVERLAP1D;
  p.inst.r1 = 0;
  p.inst.mode = k.rows > 1 ? 1 : 0;
  p.out = c->sep_tmp;
  int v = -1;
  if (choose_variant(c, p, &v) != SKEL_OK) return cudaErrorInvalidValue;
  cudaError_t e = launch_call(c, p, v);
  if (e != cudaSuccess) return e;
  Call q = k;
  q.inst.skeleton = SKEL_SK_OVERLAP1D_COL;
  q.inst.r0 = k.inst.r1;
  q.inst.r1 = 0;
  q.w1 = k.w1b;
  q.in0 = c->sep_tmp;
  if (choose_variant(c, q, &v) != SKEL_OK) return cudaErrorInvalidValue;
  return launch_call(c, q, v);
}

cudaError_t launch_call(skel_ctx* c, const Call& k, int v) {
  Launch L{c->stream, c->sms, &c->launches, c->tile_ctr, &c->tile_next};
  const skel_instance& i = k.inst;
  switch (i.skeleton) {
    case SKEL_SK_REDUCE_ROWS:
      return launch_reduce_rows(L, v, i.dtype, i.fn, k.in0, k.rows, k.cols, k.out);
    case SKEL_SK_SEPARABLE:
      if (v == 0) return launch_separable_two_pass(c, k);
      return launch_separable_fused(L, v, k.w1, k.w1b, i.r0, i.r1, i.edge, k.pad, static_cast<const float*>(k.in0),
                                    static_cast<float*>(k.out), k.rows, k.cols);
    case SKEL_SK_MAP:
      if (i.fn == SKEL_FN_MULADD) return launch_map3(L, v, i.dtype, k.in0, k.in1, k.in2, k.out, k.n);
      return launch_map(L, v, i.dtype, i.fn, i.mode != 0, k.cbits, k.in0, k.in1, k.out, k.n);
    case SKEL_SK_REDUCE:
      return launch_mapreduce(L, c->scratch, v, i.dtype, FN_IDENT_, false, i.fn, 0, k.in0, nullptr, k.n, k.out, c->reverse_next);
    case SKEL_SK_MAPREDUCE:
      return launch_mapreduce(L, c->scratch, v, i.dtype, i.fn, i.mode != 0, i.fn2, k.cbits, k.in0, k.in1, k.n, k.out, c->reverse_next);
    case SKEL_SK_SCAN:
      return launch_scan(L, c->scratch, v, i.dtype, i.fn, i.mode == SKEL_SCAN_EXCLUSIVE, k.cbits, k.in0, k.out, k.n);
    case SKEL_SK_OVERLAP1D:
      return launch_overlap1d_rows(L, v, i.dtype, k.w1, i.r0, i.edge, k.pad, static_cast<const float*>(k.in0),
                                   static_cast<float*>(k.out), k.rows, k.cols);
    case SKEL_SK_OVERLAP1D_COL:
      return launch_overlap1d_cols(L, v, i.dtype, k.w1, i.r0, i.edge, k.pad, static_cast<const float*>(k.in0),
                                   static_cast<float*>(k.out), k.rows, k.cols);
    case SKEL_SK_OVERLAP2D:
      return launch_overlap2d(L, v, i.dtype, k.w2, i.r0, i.r1, i.edge, k.pad, static_cast<const float*>(k.in0),
                              static_cast<float*>(k.out), k.rows, k.cols);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_call_f64(skel_ctx* c, const Call& k) {
  Launch L{c->stream, c->sms, &c->launches, c->tile_ctr, &c->tile_next};
  const skel_instance& i = k.inst;
  const double* in0 = static_cast<const double*>(k.in0);
  const double* in1 = static_cast<const double*>(k.in1);
  double* out = static_cast<double*>(k.out);
  switch (i.skeleton) {
    case SKEL_SK_MAP:
      return launch_map_f64(L, i.fn, i.mode != 0, k.c64, in0, in1, static_cast<const double*>(k.in2), out, k.n);
    case SKEL_SK_REDUCE:
      return launch_mapreduce_f64(L, c->scratch, FN_IDENT_, false, i.fn, 0.0, in0, nullptr, k.n, out);
    case SKEL_SK_MAPREDUCE:
      return launch_mapreduce_f64(L, c->scratch, i.fn, i.mode != 0, i.fn2, k.c64, in0, in1, k.n, out);
    case SKEL_SK_SCAN:
      return launch_scan_f64(L, c->scratch, i.fn, i.mode == SKEL_SCAN_EXCLUSIVE, k.c64, in0, out, k.n);
    case SKEL_SK_OVERLAP1D:
      return k.w1_64 ? launch_overlap1d_f64(L, *k.w1_64, i.r0, i.edge, k.pad64, 0, in0, out, k.rows, k.cols) : cudaErrorInvalidValue;
    case SKEL_SK_OVERLAP1D_COL:
      return k.w1_64 ? launch_overlap1d_f64(L, *k.w1_64, i.r0, i.edge, k.pad64, 1, in0, out, k.rows, k.cols) : cudaErrorInvalidValue;
    case SKEL_SK_OVERLAP2D:
      return k.w2_64 ? launch_overlap2d_f64(L, *k.w2_64, i.r0, i.r1, i.edge, k.pad64, in0, out, k.rows, k.cols) : cudaErrorInvalidValue;
  }
  return cudaErrorInvalidValue;
}

// choose + launch + bookkeeping
cudaError_t launch_call_f64(skel_ctx* c, const Call& k);

skel_status launch_now(skel_ctx* c, const Call& k) {
  if (k.inst.dtype == SKEL_F64) {  // one kernel per skeleton (f64.cu): nothing to select
    if (c->forced[k.inst.skeleton] > 0) return fail(c, SKEL_ERR_UNSUPPORTED, "fp64 elements have one variant (0) per skeleton");
    if (k.inst.skeleton == SKEL_SK_SCAN) {
      skel_status st64 = ensure_scan_state64(c, k.n);
      if (st64 != SKEL_OK) return st64;
    }
    cudaError_t e = launch_call_f64(c, k);
    if (e != cudaSuccess) return cuda_fail(c, e, "kernel launch (fp64)");
    c->last_sk = k.inst.skeleton;
    c->last_var = 0;
    return SKEL_OK;
  }
  int v = -1;
  skel_status st = choose_variant(c, k, &v);
  if (st != SKEL_OK) return st;
  if (k.inst.skeleton == SKEL_SK_SCAN) {
    st = ensure_scan_state(c, k.n);
    if (st != SKEL_OK) return st;
  }
  // L2-aware traversal (skel_ctx_set_l2_reuse): a kernel that streams an operand front to back leaves the operand's
  // TAIL in the 126 MB L2. When the launch right before this one read the same operand in one direction, a Reduce /
  // MapReduce walks it in the other, so its first chunks are L2 hits instead of HBM reads (a forward walk would evict
  // those lines before reaching them). Same result bits either way (reduce.cu); other kernels always walk forward.
  const bool red = k.inst.skeleton == SKEL_SK_REDUCE || k.inst.skeleton == SKEL_SK_MAPREDUCE;
  c->reverse_next = red && c->l2_reuse && c->walk_in0 == k.in0 && c->walk_launch == c->stats.launches + uint64_t(c->launches) && !c->walk_reverse;
  cudaError_t e = launch_call(c, k, v);
  const bool reversed = c->reverse_next;
  c->reverse_next = false;
  if (e != cudaSuccess) return cuda_fail(c, e, "kernel launch");
  c->walk_in0 = k.in0;
  c->walk_reverse = reversed;
  c->walk_launch = c->stats.launches + uint64_t(c->launches);
  c->last_sk = k.inst.skeleton;
  c->last_var = v;
  return SKEL_OK;
}

// ---- cross-call fusion ----------------------------------------------------------
// With fusion enabled, the LAUNCH of a call that can be part of the chain
//   Map(f in {ADD, MULT, MAX}, constant c, f32 vector) -> MapOverlap1D(vector) -> Reduce(ADD | MAX)
// is held back (coherence bookkeeping and transfers happen at call time as always; every launch is
// on one in-order stream, so delaying a launch behind nothing but bookkeeping changes no result).
// The chain is launched as ONE kernel (fused.cu) when its Reduce arrives, or call by call when
// anything else happens first: every entry point that touches the stream flushes.
int chain_kind(const skel_ctx* c, const Call& k) {
  const skel_instance& i = k.inst;
  if (i.skeleton < 0 || i.skeleton >= SKEL_SK_COUNT || c->forced[i.skeleton] >= 0 || k.n == 0) return 0;
  if (i.skeleton == SKEL_SK_MAP && i.dtype == SKEL_F32 && i.mode == 0 &&
      (i.fn == SKEL_FN_ADD || i.fn == SKEL_FN_MULT || i.fn == SKEL_FN_MAX))
    return 1;
  if (i.skeleton == SKEL_SK_OVERLAP1D && i.dtype == SKEL_F32 && k.rows == 1 && i.r0 >= 0 && i.r0 <= 8) return 2;
  if (i.skeleton == SKEL_SK_REDUCE && i.dtype == SKEL_F32 && (i.fn == SKEL_FN_ADD || i.fn == SKEL_FN_MAX)) return 3;
  return 0;
}

bool has_pending(const skel_ctx* c) { return !c->pending.empty(); }

skel_status flush_pending(skel_ctx* c) {
  if (c->pending.empty()) return SKEL_OK;
  std::vector<PendingCall> q;
  q.swap(c->pending);
  const Call* map = nullptr;
  const Call* ov = nullptr;
  const Call* red = nullptr;
  for (const PendingCall& p : q) {
    const int kind = chain_kind(c, p.k);
    if (kind == 1) map = &p.k;
    if (kind == 2) ov = &p.k;
    if (kind == 3) red = &p.k;
  }
  skel_status st = SKEL_OK;
  // a Reduce whose result lands inside a container the chain itself writes keeps the call-by-call order
  // (the in-place Map's buffer may be swapped under it)
  const bool result_in_chain = red && red->out_st && ((map && red->out_st == map->out_st) || (ov && red->out_st == ov->out_st));
  if (ov && (map || red) && !result_in_chain) {
    const float* in = static_cast<const float*>(map ? map->in0 : ov->in0);
    float* map_out = map ? static_cast<float*>(map->out) : nullptr;
    bool swap = false;
    if (map && map->out == map->in0) {  // in place: A' goes to the spare buffer, which then becomes A's
      Storage* a = map->out_st;
      const size_t bytes = a->n * esize(a->dtype);
      if (a->dev_owned) {
        if (c->spare && c->spare_bytes != bytes) {
          dev_free(c, c->spare);
          c->spare = nullptr;
        }
        if (!c->spare && dev_alloc(c, bytes, &c->spare) == SKEL_OK) c->spare_bytes = bytes;
        if (c->spare) {
          map_out = static_cast<float*>(c->spare);
          swap = true;
        }
      }
    }
    const int map_fn = map ? map->inst.fn : FN_IDENT_;
    const int red_op = red ? red->inst.fn : FUSED_NO_REDUCE;
    if (fused_chain_ok(map_fn, ov->inst.r0, red_op, in, map_out, ov->out, ov->n)) {
      Launch L{c->stream, c->sms, &c->launches, c->tile_ctr, &c->tile_next};
      cudaError_t e = launch_fused_chain(L, c->scratch, map_fn, map ? map->cbits : 0u, ov->w1, ov->inst.r0, ov->inst.edge,
                                         ov->pad, red_op, in, map_out, static_cast<float*>(ov->out), ov->n,
                                         red ? static_cast<float*>(red->out) : nullptr);
      if (e != cudaSuccess) return cuda_fail(c, e, "fused chain launch");
      if (swap) {
        Storage* a = map->out_st;
        void* old = a->dev;
        a->dev = c->spare;
        c->spare = old;
      }
      c->last_sk = ov->inst.skeleton;
      c->last_var = -2;  // "fused"
      c->stats.fused_launches += 1;
      c->stats.fused_calls += q.size();
      c->stats.launches += c->launches;
      c->launches = 0;
      return mark_enqueued(c);
    }
  }
  for (const PendingCall& p : q) {
    st = launch_now(c, p.k);
    if (st != SKEL_OK) return st;
  }
  c->stats.launches += c->launches;
  c->launches = 0;
  return mark_enqueued(c);
}

void record_call(skel_ctx* c, const OperandSet& set) {
  if (c->recorded.empty() || c->recorded.back().variant != -1000) return;  // run_call left a slot only when recording
  c->recorded.back().set = set;
  c->recorded.back().variant = c->last_var;
}

skel_status run_call(skel_ctx* c, const Call& k) {
  if (c->recording) {
    if (c->fusion) return fail(c, SKEL_ERR_UNSUPPORTED, "skel_replay_begin: recording needs cross-call fusion off");
    c->recorded.push_back(RecordedCall{k, OperandSet{}, -1000});
  }
  if (!c->fusion) return launch_now(c, k);
  const int kind = chain_kind(c, k);
  bool extends = false;
  if (!c->pending.empty()) {
    const Call& last = c->pending.back().k;
    const int lk = chain_kind(c, last);
    extends = (lk == 1 && kind == 2 && k.in0 == last.out && k.n == last.n) ||
              (lk == 2 && kind == 3 && k.in0 == last.out && k.n == last.n);
  }
  if (!extends) {
    skel_status st = flush_pending(c);
    if (st != SKEL_OK) return st;
  }
  if (kind == 1 || kind == 2 || (kind == 3 && extends)) {
    c->pending.push_back(PendingCall{k});
    if (kind == 3) return flush_pending(c);  // the chain is complete
    return SKEL_OK;
  }
  return launch_now(c, k);
}

bool red_op_ok(int op) { return op == SKEL_FN_ADD || op == SKEL_FN_MULT || op == SKEL_FN_MAX; }
bool map_fn_ok(int f) { return f == SKEL_FN_ADD || f == SKEL_FN_MULT || f == SKEL_FN_MAX || f == SKEL_FN_SAXPY; }

// convert the scalar constant to the element type's bits
skel_status const_bits(skel_ctx* c, int dtype, double v, uint32_t* bits) {
  if (dtype == SKEL_F64) {  // the constant travels as a double (Call::c64)
    *bits = 0;
    return SKEL_OK;
  }
  if (dtype == SKEL_F32) {
    const float f = static_cast<float>(v);
    memcpy(bits, &f, 4);
    return SKEL_OK;
  }
  if (!(v >= -2147483648.0 && v <= 2147483647.0) || v != floor(v))
    return fail(c, SKEL_ERR_INVALID_ARG, "constant is not an int32 value");
  const int32_t i = static_cast<int32_t>(v);
  memcpy(bits, &i, 4);
  return SKEL_OK;
}

skel_status scalar_to_host(skel_ctx* c, int dtype, void* host_result) {
  skel_status fst = flush_pending(c);
  if (fst != SKEL_OK) return fst;
  // zero-copy: the kernel's last block wrote the scalar into the mapped host slot (no device-to-host copy to
  // enqueue and wait for); visible to the host once the event recorded after the reducing kernel has fired
  skel_status wst = wait_seq(c, c->seq);
  if (wst != SKEL_OK) return wst;
  memcpy(host_result, c->h_result, esize(dtype));
  c->stats.scalar_d2h_count += 1;
  return SKEL_OK;
}

skel_status mapreduce_impl(skel_ctx* c, bool plain_reduce, int map_f, int red_op, double cval, const skel_vector* in0,
                           const skel_vector* in1, void* host_result, skel_vector* out, size_t out_index,
                           skel_future** fut = nullptr) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (fut) *fut = nullptr;
  if (!vec_ok(in0) || (in1 && !vec_ok(in1))) return fail(c, SKEL_ERR_INVALID_ARG, "bad input handle");
  if (!host_result && !fut && !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "no result destination");
  if (!red_op_ok(red_op)) return fail(c, SKEL_ERR_UNSUPPORTED, "reduce operator must be ADD, MULT or MAX");
  if (!plain_reduce && !map_fn_ok(map_f)) return fail(c, SKEL_ERR_UNSUPPORTED, "map function must be ADD, MULT, MAX or SAXPY");
  if (!plain_reduce && map_f == SKEL_FN_SAXPY && !in1) return fail(c, SKEL_ERR_INVALID_ARG, "SAXPY needs in1");
  Storage* a = in0->st;
  Storage* b = in1 ? in1->st : nullptr;
  if (b && b->dtype != a->dtype) return fail(c, SKEL_ERR_DTYPE, "operand element types differ");
  if (b && b->n != a->n) return fail(c, SKEL_ERR_SIZE_MISMATCH, "operand sizes differ");
  if (out) {
    if (out->st->dtype != a->dtype) return fail(c, SKEL_ERR_DTYPE, "result element type differs");
    if (out_index >= out->st->n) return fail(c, SKEL_ERR_INVALID_ARG, "out_index out of range");
    if (out->st == a || out->st == b) return fail(c, SKEL_ERR_ALIAS, "result vector aliases an input");
  }
  if (a->n == 0) return fail(c, SKEL_ERR_EMPTY, "reduce of an empty vector");
  Call k;
  k.inst.skeleton = plain_reduce ? SKEL_SK_REDUCE : SKEL_SK_MAPREDUCE;
  k.inst.fn = plain_reduce ? red_op : map_f;
  k.inst.fn2 = plain_reduce ? 0 : red_op;
  k.inst.dtype = a->dtype;
  k.inst.mode = b ? 1 : 0;
  skel_status st = SKEL_OK;
  if (!plain_reduce) {
    st = const_bits(c, a->dtype, cval, &k.cbits);
    if (st != SKEL_OK) return st;
    k.c64 = cval;
  }
  OperandSet set;
  set.add(a, ACC_READ);
  if (b) set.add(b, ACC_READ);
  if (out) set.add(out->st, (out->st->n == 1 || out->st->state == ST_UNINIT) ? ACC_WRITE : ACC_READWRITE);
  st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  int slot = -1;
  if (fut) {  // a pinned, mapped 8-byte slot of the context's pool for this result
    if (!c->h_slots) {
      CU(c, cudaHostAlloc(&c->h_slots, size_t(FUTURE_SLOTS) * 8, cudaHostAllocMapped));
      CU(c, cudaHostGetDevicePointer(&c->h_slots_dev, c->h_slots, 0));
      for (int i = FUTURE_SLOTS - 1; i >= 0; --i) c->free_slots.push_back(i);
    }
    if (c->free_slots.empty()) return fail(c, SKEL_ERR_BUSY, "too many outstanding futures (destroy some)");
    slot = c->free_slots.back();
  }
  k.in0 = a->dev;
  k.in1 = b ? b->dev : nullptr;
  k.n = a->n;
  k.out = out ? static_cast<void*>(static_cast<char*>(out->st->dev) + out_index * esize(a->dtype))
              : (fut ? static_cast<void*>(static_cast<char*>(c->h_slots_dev) + size_t(slot) * 8) : c->h_result_dev);
  k.in_st = a;
  k.out_st = out ? out->st : nullptr;
  st = run_call(c, k);
  if (st != SKEL_OK) return st;
  st = publish_all(c, set);
  if (st != SKEL_OK) return st;
  if (fut) {
    skel_future* f = new (std::nothrow) skel_future{MAGIC_FUT, c, slot, a->dtype, c->seq};
    if (!f) return fail(c, SKEL_ERR_OOM, "host allocation failed");
    c->free_slots.pop_back();
    ++c->live;
    *fut = f;
    return SKEL_OK;
  }
  if (host_result) return scalar_to_host(c, a->dtype, host_result);
  return SKEL_OK;
}

skel_status overlap_check(skel_ctx* c, const Handle* in, const Handle* out, int edge, int dtype = SKEL_F32) {
  if (in->st->dtype != dtype || out->st->dtype != dtype)
    return fail(c, SKEL_ERR_DTYPE, dtype == SKEL_F32   ? "skel_mapoverlap_*: f32 containers expected (int32: *_i32, fp64: *_f64)"
                                   : dtype == SKEL_I32 ? "skel_mapoverlap_*_i32: int32 containers expected"
                                                       : "skel_mapoverlap_*_f64: fp64 containers expected");
  if (in->rows != out->rows || in->cols != out->cols) return fail(c, SKEL_ERR_SIZE_MISMATCH, "input and output shapes differ");
  if (in->st == out->st) return fail(c, SKEL_ERR_ALIAS, "MapOverlap output must not alias its input");
  if (edge != SKEL_EDGE_CONSTANT && edge != SKEL_EDGE_DUPLICATE && edge != SKEL_EDGE_CYCLIC) return fail(c, SKEL_ERR_INVALID_ARG, "bad edge policy");
  return SKEL_OK;
}

skel_status overlap_run(skel_ctx* c, Call& k, const Handle* in, Handle* out) {
  OperandSet set;
  set.add(in->st, ACC_READ);
  set.add(out->st, ACC_WRITE);
  skel_status st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  k.in0 = in->st->dev;
  k.out = out->st->dev;
  k.n = in->st->n;
  k.in_st = in->st;
  k.out_st = out->st;
  st = run_call(c, k);
  if (st != SKEL_OK) return st;
  return publish_all(c, set);
}

}  // namespace

// =================================================================================================
#pragma GCC visibility push(default)
extern "C" {

int skel_abi_version(void) { return SKEL_ABI_VERSION; }

skel_status skel_ctx_create(void* cuda_stream, skel_alloc_fn alloc, skel_free_fn free_, void* user, skel_ctx** out) {
  if (!out) return SKEL_ERR_INVALID_ARG;
  *out = nullptr;
  if ((alloc == nullptr) != (free_ == nullptr)) return SKEL_ERR_INVALID_ARG;
  skel_ctx* c = new (std::nothrow) skel_ctx;
  if (!c) return SKEL_ERR_OOM;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->alloc = alloc;
  c->free_ = free_;
  c->user = user;
  for (int i = 0; i < SKEL_SK_COUNT; ++i) c->forced[i] = -1;
  const char* env = getenv("SKEL_COHERENCE");
  if (env && strcmp(env, "eager") == 0) c->mode = MODE_EAGER;
  const char* plan = getenv("SKEL_PLAN_FILE");
  if (plan && *plan && !c->plan.load(plan))  // the context is usable (untuned defaults); skel_last_error says why
    c->err = std::string("SKEL_PLAN_FILE: cannot read or parse '") + plan + "'; running with the built-in defaults";
  *out = c;
  return SKEL_OK;
}

skel_status skel_ctx_destroy(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (c->live > 0) return fail(c, SKEL_ERR_BUSY, "containers or futures of this context are still alive");
  if (c->dev_ready) {
    flush_pending(c);
    cudaStreamSynchronize(c->stream);
    if (c->copy_stream) {
      cudaStreamSynchronize(c->copy_stream);
      cudaStreamDestroy(c->copy_stream);
    }
    if (c->spare) dev_free(c, c->spare);
    if (c->sep_tmp) dev_free(c, c->sep_tmp);
    cudaFree(c->scratch.partials);
    if (c->scratch.scan_state) cudaFree(c->scratch.scan_state);
    if (c->scratch.scan_state64) cudaFree(c->scratch.scan_state64);
    cudaFreeHost(c->h_result);
    if (c->h_slots) cudaFreeHost(c->h_slots);
    for (cudaEvent_t e : c->ring.ev)
      if (e) cudaEventDestroy(e);
  }
  c->magic = 0;
  delete c;
  return SKEL_OK;
}

skel_status skel_ctx_sync(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (c->sticky) return SKEL_ERR_CUDA;
  if (!c->dev_ready) return SKEL_OK;
  skel_status st = flush_pending(c);
  if (st != SKEL_OK) return st;
  CU(c, cudaStreamSynchronize(c->stream));
  if (c->copy_stream) CU(c, cudaStreamSynchronize(c->copy_stream));  // prefetch downloads in flight
  c->done_seq = c->seq;
  return SKEL_OK;
}

skel_status skel_ctx_set_l2_reuse(skel_ctx* c, int enable) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  c->l2_reuse = enable != 0;
  return SKEL_OK;
}

skel_status skel_ctx_set_fusion(skel_ctx* c, int enable) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  skel_status st = flush_pending(c);
  c->fusion = enable != 0;
  return st;
}

skel_status skel_ctx_flush(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  return flush_pending(c);
}

skel_status skel_ctx_set_coherence(skel_ctx* c, skel_coherence mode) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (mode != SKEL_LAZY && mode != SKEL_EAGER) return fail(c, SKEL_ERR_INVALID_ARG, "bad coherence mode");
  skel_status st = flush_pending(c);
  if (st != SKEL_OK) return st;
  c->mode = mode;
  return SKEL_OK;
}

const char* skel_last_error(skel_ctx* c) { return ctx_ok(c) ? c->err.c_str() : "invalid context"; }

// ---- vectors ------------------------------------------------------------------------------------
skel_status skel_vector_create(skel_ctx* c, skel_dtype dt, size_t n, skel_vector** out) {
  return make_handle<skel_vector>(c, MAGIC_VEC, dt, 1, n, out);
}

skel_status skel_vector_create_from(skel_ctx* c, skel_dtype dt, size_t n, const void* src, skel_vector** out) {
  skel_status st = make_handle<skel_vector>(c, MAGIC_VEC, dt, 1, n, out);
  if (st != SKEL_OK) return st;
  st = fill_from(c, (*out)->st, src);
  if (st != SKEL_OK) {
    release_handle(*out);
    delete *out;
    *out = nullptr;
  }
  return st;
}

skel_status skel_vector_adopt_device(skel_ctx* c, skel_dtype dt, size_t n, void* dptr, skel_vector** out) {
  if (ctx_ok(c) && n > 0 && !dptr) return fail(c, SKEL_ERR_INVALID_ARG, "dptr is NULL");
  skel_status st = make_handle<skel_vector>(c, MAGIC_VEC, dt, 1, n, out);
  if (st != SKEL_OK) return st;
  (*out)->st->dev = dptr;
  (*out)->st->dev_owned = false;
  (*out)->st->state = ST_DEVICE;
  return SKEL_OK;
}

skel_status skel_vector_destroy(skel_vector* v) {
  if (!vec_ok(v)) return SKEL_ERR_INVALID_ARG;
  skel_status st = release_handle(v);
  if (st == SKEL_OK) delete v;
  return st;
}

skel_status skel_vector_size(const skel_vector* v, size_t* n) {
  if (!vec_ok(v) || !n) return SKEL_ERR_INVALID_ARG;
  *n = v->st->n;
  return SKEL_OK;
}

skel_status skel_vector_host_acquire(skel_vector* v, skel_access mode, void** host_ptr) {
  if (!vec_ok(v)) return SKEL_ERR_INVALID_ARG;
  return host_acquire(v, mode, host_ptr);
}

skel_status skel_vector_host_acquire_range(skel_vector* v, skel_access mode, size_t offset, size_t count, void** host_ptr) {
  if (!vec_ok(v)) return SKEL_ERR_INVALID_ARG;
  return host_acquire_range(v, mode, offset, count, host_ptr);
}

skel_status skel_vector_prefetch_host(skel_vector* v) {
  if (!vec_ok(v)) return SKEL_ERR_INVALID_ARG;
  return prefetch_host(v);
}

skel_status skel_vector_host_release(skel_vector* v) {
  if (!vec_ok(v)) return SKEL_ERR_INVALID_ARG;
  return host_release(v);
}

skel_status skel_vector_device_ptr(const skel_vector* v, void** dptr, int* valid) {
  if (!vec_ok(v) || !dptr) return SKEL_ERR_INVALID_ARG;
  flush_pending(v->st->ctx);  // the caller is about to use the stream / the pointer (a fused in-place Map swaps buffers)
  upload_host_newer(v->st->ctx, v->st);
  *dptr = v->st->dev;
  if (valid) *valid = (v->st->state & 2) ? 1 : 0;
  return SKEL_OK;
}

skel_status skel_vector_state(const skel_vector* v, int* state) {
  if (!vec_ok(v) || !state) return SKEL_ERR_INVALID_ARG;
  *state = v->st->state;
  return SKEL_OK;
}

// ---- matrices -----------------------------------------------------------------------------------
skel_status skel_matrix_create(skel_ctx* c, skel_dtype dt, size_t rows, size_t cols, skel_matrix** out) {
  return make_handle<skel_matrix>(c, MAGIC_MAT, dt, rows, cols, out);
}

skel_status skel_matrix_create_from(skel_ctx* c, skel_dtype dt, size_t rows, size_t cols, const void* src, skel_matrix** out) {
  skel_status st = make_handle<skel_matrix>(c, MAGIC_MAT, dt, rows, cols, out);
  if (st != SKEL_OK) return st;
  st = fill_from(c, (*out)->st, src);
  if (st != SKEL_OK) {
    release_handle(*out);
    delete *out;
    *out = nullptr;
  }
  return st;
}

skel_status skel_matrix_adopt_device(skel_ctx* c, skel_dtype dt, size_t rows, size_t cols, void* dptr, skel_matrix** out) {
  if (ctx_ok(c) && rows * cols > 0 && !dptr) return fail(c, SKEL_ERR_INVALID_ARG, "dptr is NULL");
  skel_status st = make_handle<skel_matrix>(c, MAGIC_MAT, dt, rows, cols, out);
  if (st != SKEL_OK) return st;
  (*out)->st->dev = dptr;
  (*out)->st->dev_owned = false;
  (*out)->st->state = ST_DEVICE;
  return SKEL_OK;
}

skel_status skel_matrix_destroy(skel_matrix* m) {
  if (!mat_ok(m)) return SKEL_ERR_INVALID_ARG;
  skel_status st = release_handle(m);
  if (st == SKEL_OK) delete m;
  return st;
}

skel_status skel_matrix_shape(const skel_matrix* m, size_t* rows, size_t* cols) {
  if (!mat_ok(m) || !rows || !cols) return SKEL_ERR_INVALID_ARG;
  *rows = m->rows;
  *cols = m->cols;
  return SKEL_OK;
}

skel_status skel_matrix_host_acquire(skel_matrix* m, skel_access mode, void** host_ptr) {
  if (!mat_ok(m)) return SKEL_ERR_INVALID_ARG;
  return host_acquire(m, mode, host_ptr);
}

skel_status skel_matrix_host_acquire_rows(skel_matrix* m, skel_access mode, size_t row0, size_t nrows, void** host_ptr) {
  if (!mat_ok(m)) return SKEL_ERR_INVALID_ARG;
  if (row0 > m->rows || nrows > m->rows - row0) return fail(m->st->ctx, SKEL_ERR_INVALID_ARG, "row range out of bounds");
  return host_acquire_range(m, mode, row0 * m->cols, nrows * m->cols, host_ptr);
}

skel_status skel_matrix_prefetch_host(skel_matrix* m) {
  if (!mat_ok(m)) return SKEL_ERR_INVALID_ARG;
  return prefetch_host(m);
}

skel_status skel_matrix_host_release(skel_matrix* m) {
  if (!mat_ok(m)) return SKEL_ERR_INVALID_ARG;
  return host_release(m);
}

skel_status skel_matrix_as_vector(skel_matrix* m, skel_vector** view) {
  if (!mat_ok(m) || !view) return SKEL_ERR_INVALID_ARG;
  skel_vector* v = new (std::nothrow) skel_vector;
  if (!v) return fail(m->st->ctx, SKEL_ERR_OOM, "host allocation failed");
  v->magic = MAGIC_VEC;
  v->st = m->st;
  v->rows = 1;
  v->cols = m->st->n;
  ++m->st->refs;
  ++m->st->ctx->live;
  *view = v;
  return SKEL_OK;
}

// ---- Map ------------------------------------------------------------------------------------------
skel_status skel_map(skel_ctx* c, skel_fn f, double cval, const skel_vector* in0, const skel_vector* in1, skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in0) || (in1 && !vec_ok(in1)) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad vector handle");
  if (!map_fn_ok(f)) return fail(c, SKEL_ERR_UNSUPPORTED, "map function must be ADD, MULT, MAX or SAXPY");
  if (f == SKEL_FN_SAXPY && !in1) return fail(c, SKEL_ERR_INVALID_ARG, "SAXPY needs in1");
  Storage* a = in0->st;
  Storage* b = in1 ? in1->st : nullptr;
  Storage* o = out->st;
  if ((b && b->dtype != a->dtype) || o->dtype != a->dtype) return fail(c, SKEL_ERR_DTYPE, "operand element types differ");
  if ((b && b->n != a->n) || o->n != a->n) return fail(c, SKEL_ERR_SIZE_MISMATCH, "operand sizes differ");
  Call k;
  k.inst.skeleton = SKEL_SK_MAP;
  k.inst.fn = f;
  k.inst.dtype = a->dtype;
  k.inst.mode = b ? 1 : 0;
  k.c64 = cval;
  skel_status st = const_bits(c, a->dtype, cval, &k.cbits);
  if (st != SKEL_OK) return st;
  OperandSet set;
  set.add(a, ACC_READ);
  if (b) set.add(b, ACC_READ);
  set.add(o, ACC_WRITE);
  st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  k.in0 = a->dev;
  k.in1 = b ? b->dev : nullptr;
  k.out = o->dev;
  k.n = a->n;
  k.in_st = a;
  k.out_st = o;
  if (k.n > 0) {
    st = run_call(c, k);
    if (st != SKEL_OK) return st;
  }
  return publish_all(c, set);
}

skel_status skel_map3(skel_ctx* c, skel_fn f, const skel_vector* in0, const skel_vector* in1, const skel_vector* in2,
                      skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in0) || !vec_ok(in1) || !vec_ok(in2) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad vector handle");
  if (f != SKEL_FN_MULADD) return fail(c, SKEL_ERR_UNSUPPORTED, "the three-vector map function must be MULADD");
  Storage *a = in0->st, *b = in1->st, *d = in2->st, *o = out->st;
  if (b->dtype != a->dtype || d->dtype != a->dtype || o->dtype != a->dtype) return fail(c, SKEL_ERR_DTYPE, "operand element types differ");
  if (b->n != a->n || d->n != a->n || o->n != a->n) return fail(c, SKEL_ERR_SIZE_MISMATCH, "operand sizes differ");
  Call k;
  k.inst.skeleton = SKEL_SK_MAP;
  k.inst.fn = f;
  k.inst.dtype = a->dtype;
  k.inst.mode = 2;  // three vectors
  OperandSet set;
  set.add(a, ACC_READ);
  set.add(b, ACC_READ);
  set.add(d, ACC_READ);
  set.add(o, ACC_WRITE);
  skel_status st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  k.in0 = a->dev;
  k.in1 = b->dev;
  k.in2 = d->dev;
  k.out = o->dev;
  k.n = a->n;
  k.in_st = a;
  k.out_st = o;
  if (k.n > 0) {
    st = run_call(c, k);
    if (st != SKEL_OK) return st;
  }
  return publish_all(c, set);
}

// ---- Reduce / MapReduce ---------------------------------------------------------------------------
skel_status skel_reduce(skel_ctx* c, skel_fn op, const skel_vector* in, void* host_result) {
  if (ctx_ok(c) && !host_result) return fail(c, SKEL_ERR_INVALID_ARG, "host_result is NULL");
  return mapreduce_impl(c, true, 0, op, 0.0, in, nullptr, host_result, nullptr, 0);
}

skel_status skel_reduce_to(skel_ctx* c, skel_fn op, const skel_vector* in, skel_vector* out, size_t out_index) {
  if (ctx_ok(c) && !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad result vector");
  return mapreduce_impl(c, true, 0, op, 0.0, in, nullptr, nullptr, out, out_index);
}

skel_status skel_mapreduce(skel_ctx* c, skel_fn map_f, skel_fn red_op, double cval, const skel_vector* in0,
                           const skel_vector* in1, void* host_result) {
  if (ctx_ok(c) && !host_result) return fail(c, SKEL_ERR_INVALID_ARG, "host_result is NULL");
  return mapreduce_impl(c, false, map_f, red_op, cval, in0, in1, host_result, nullptr, 0);
}

skel_status skel_mapreduce_to(skel_ctx* c, skel_fn map_f, skel_fn red_op, double cval, const skel_vector* in0,
                              const skel_vector* in1, skel_vector* out, size_t out_index) {
  if (ctx_ok(c) && !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad result vector");
  return mapreduce_impl(c, false, map_f, red_op, cval, in0, in1, nullptr, out, out_index);
}

skel_status skel_reduce_async(skel_ctx* c, skel_fn op, const skel_vector* in, skel_future** out) {
  if (ctx_ok(c) && !out) return fail(c, SKEL_ERR_INVALID_ARG, "out is NULL");
  return mapreduce_impl(c, true, 0, op, 0.0, in, nullptr, nullptr, nullptr, 0, out);
}

skel_status skel_mapreduce_async(skel_ctx* c, skel_fn map_f, skel_fn red_op, double cval, const skel_vector* in0,
                                 const skel_vector* in1, skel_future** out) {
  if (ctx_ok(c) && !out) return fail(c, SKEL_ERR_INVALID_ARG, "out is NULL");
  return mapreduce_impl(c, false, map_f, red_op, cval, in0, in1, nullptr, nullptr, 0, out);
}

skel_status skel_future_wait(skel_future* f, void* host_result) {
  if (!f || f->magic != MAGIC_FUT) return SKEL_ERR_INVALID_ARG;
  skel_ctx* c = f->ctx;
  if (!host_result) return fail(c, SKEL_ERR_INVALID_ARG, "host_result is NULL");
  if (c->sticky) return SKEL_ERR_CUDA;
  skel_status st = wait_seq(c, f->seq);  // the event recorded after the reducing kernel, not the whole stream
  if (st != SKEL_OK) return st;
  memcpy(host_result, static_cast<char*>(c->h_slots) + size_t(f->slot) * 8, esize(f->dtype));
  c->stats.scalar_d2h_count += 1;
  return SKEL_OK;
}

skel_status skel_future_ready(skel_future* f, int* ready) {
  if (!f || f->magic != MAGIC_FUT) return SKEL_ERR_INVALID_ARG;
  skel_ctx* c = f->ctx;
  if (!ready) return fail(c, SKEL_ERR_INVALID_ARG, "ready is NULL");
  *ready = 0;
  if (f->seq <= c->done_seq) {
    *ready = 1;
    return SKEL_OK;
  }
  skel_status st = flush_pending(c);
  if (st != SKEL_OK) return st;
  st = mark_enqueued(c);
  if (st != SKEL_OK) return st;
  const EventRing& r = c->ring;
  int best = -1;
  for (int i = 0; i < EventRing::N; ++i)
    if (r.ev[i] && r.seq[i] >= f->seq && (best < 0 || r.seq[i] < r.seq[best])) best = i;
  if (best < 0) return SKEL_OK;
  const cudaError_t e = cudaEventQuery(r.ev[best]);
  if (e == cudaSuccess) {
    if (r.seq[best] > c->done_seq) c->done_seq = r.seq[best];
    *ready = 1;
  } else if (e != cudaErrorNotReady) {
    return cuda_fail(c, e, "cudaEventQuery");
  }
  return SKEL_OK;
}

skel_status skel_future_destroy(skel_future* f) {
  if (!f || f->magic != MAGIC_FUT) return SKEL_ERR_INVALID_ARG;
  skel_ctx* c = f->ctx;
  if (!c->sticky) wait_seq(c, f->seq);  // the kernel may still be about to write the slot
  c->free_slots.push_back(f->slot);
  --c->live;
  f->magic = 0;
  delete f;
  return SKEL_OK;
}

skel_status skel_reduce_rows(skel_ctx* c, skel_fn op, const skel_matrix* in, skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  if (!red_op_ok(op)) return fail(c, SKEL_ERR_UNSUPPORTED, "reduce operator must be ADD, MULT or MAX");
  if (out->st->dtype != in->st->dtype) return fail(c, SKEL_ERR_DTYPE, "result element type differs");
  if (in->st->dtype == SKEL_F64) return fail(c, SKEL_ERR_DTYPE, "skel_reduce_rows: f32 and i32 matrices only");
  if (out->st->n != in->rows) return fail(c, SKEL_ERR_SIZE_MISMATCH, "result vector must have one element per row");
  if (out->st == in->st) return fail(c, SKEL_ERR_ALIAS, "result vector aliases the input");
  if (in->rows > 0 && in->cols == 0) return fail(c, SKEL_ERR_EMPTY, "reduce of empty rows");
  Call k;
  k.inst.skeleton = SKEL_SK_REDUCE_ROWS;
  k.inst.fn = op;
  k.inst.dtype = in->st->dtype;
  k.rows = in->rows;
  k.cols = in->cols;
  OperandSet set;
  set.add(in->st, ACC_READ);
  set.add(out->st, ACC_WRITE);
  skel_status st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  k.in0 = in->st->dev;
  k.out = out->st->dev;
  k.n = in->st->n;
  k.in_st = in->st;
  k.out_st = out->st;
  if (in->rows > 0) {
    st = run_call(c, k);
    if (st != SKEL_OK) return st;
  }
  return publish_all(c, set);
}

// ---- MapOverlap -----------------------------------------------------------------------------------
namespace {
// dtype: SKEL_F32 (w: floats, pad rounded to f32) or SKEL_I32 (w: int32, pad an int32): 32-bit images either way
skel_status overlap1d_impl(skel_ctx* c, int dtype, const void* w, int r, skel_edge edge, uint32_t pad_bits, int axis,
                           const Handle* in, Handle* out, bool is_matrix) {
  if (!w) return fail(c, SKEL_ERR_INVALID_ARG, "NULL weights");
  if (is_matrix && axis != SKEL_AXIS_ROW && axis != SKEL_AXIS_COL) return fail(c, SKEL_ERR_INVALID_ARG, "bad axis");
  if (r < 0 || r > SKEL_MAX_RADIUS_1D) return fail(c, SKEL_ERR_UNSUPPORTED, "radius out of range");
  skel_status st = overlap_check(c, in, out, edge, dtype);
  if (st != SKEL_OK) return st;
  Call k;
  k.inst.skeleton = (!is_matrix || axis == SKEL_AXIS_ROW) ? SKEL_SK_OVERLAP1D : SKEL_SK_OVERLAP1D_COL;
  k.inst.fn = SKEL_FN_WSTENCIL;
  k.inst.dtype = dtype;
  k.inst.r0 = r;
  k.inst.edge = edge;
  k.inst.mode = (is_matrix && axis == SKEL_AXIS_ROW && in->rows > 1) ? 1 : 0;  // shape class of the plan's dispatch tree
  memcpy(&k.pad, &pad_bits, 4);
  memcpy(k.w1.w, w, 4 * size_t(2 * r + 1));
  k.rows = is_matrix ? in->rows : 1;
  k.cols = is_matrix ? in->cols : in->st->n;
  return overlap_run(c, k, in, out);
}

skel_status overlap2d_impl(skel_ctx* c, int dtype, const void* W, int ry, int rx, skel_edge edge, uint32_t pad_bits,
                           const skel_matrix* in, skel_matrix* out) {
  if (!W) return fail(c, SKEL_ERR_INVALID_ARG, "NULL weights");
  if (ry < 0 || rx < 0 || ry > SKEL_MAX_RADIUS_2D || rx > SKEL_MAX_RADIUS_2D)
    return fail(c, SKEL_ERR_UNSUPPORTED, "radius out of range");
  skel_status st = overlap_check(c, in, out, edge, dtype);
  if (st != SKEL_OK) return st;
  Call k;
  k.inst.skeleton = SKEL_SK_OVERLAP2D;
  k.inst.fn = SKEL_FN_WSTENCIL;
  k.inst.dtype = dtype;
  k.inst.r0 = ry;
  k.inst.r1 = rx;
  k.inst.edge = edge;
  memcpy(&k.pad, &pad_bits, 4);
  memcpy(k.w2.w, W, 4 * size_t(2 * ry + 1) * size_t(2 * rx + 1));
  k.rows = in->rows;
  k.cols = in->cols;
  return overlap_run(c, k, in, out);
}

skel_status overlap_f64_impl(skel_ctx* c, int skeleton, const double* w, int ry, int rx, skel_edge edge, double pad,
                             const Handle* in, Handle* out, bool is_matrix) {
  if (!w) return fail(c, SKEL_ERR_INVALID_ARG, "NULL weights");
  const bool two_d = skeleton == SKEL_SK_OVERLAP2D;
  if (two_d ? (ry < 0 || rx < 0 || ry > SKEL_MAX_RADIUS_2D || rx > SKEL_MAX_RADIUS_2D) : (ry < 0 || ry > SKEL_MAX_RADIUS_1D))
    return fail(c, SKEL_ERR_UNSUPPORTED, "radius out of range");
  skel_status st = overlap_check(c, in, out, edge, SKEL_F64);
  if (st != SKEL_OK) return st;
  Call k;
  k.inst.skeleton = skeleton;
  k.inst.fn = SKEL_FN_WSTENCIL;
  k.inst.dtype = SKEL_F64;
  k.inst.r0 = ry;
  k.inst.r1 = two_d ? rx : 0;
  k.inst.edge = edge;
  k.pad64 = pad;
  if (two_d) {
    auto p = std::make_shared<Weights2D64>();
    memcpy(p->w, w, sizeof(double) * size_t(2 * ry + 1) * size_t(2 * rx + 1));
    k.w2_64 = p;
  } else {
    auto p = std::make_shared<Weights1D64>();
    memcpy(p->w, w, sizeof(double) * size_t(2 * ry + 1));
    k.w1_64 = p;
  }
  k.rows = is_matrix ? in->rows : 1;
  k.cols = is_matrix ? in->cols : in->st->n;
  return overlap_run(c, k, in, out);
}

uint32_t f32_bits(double v) {
  const float f = static_cast<float>(v);
  uint32_t b;
  memcpy(&b, &f, 4);
  return b;
}
}  // namespace

skel_status skel_mapoverlap_1d(skel_ctx* c, const float* w, int r, skel_edge edge, double pad, const skel_vector* in,
                               skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap1d_impl(c, SKEL_F32, w, r, edge, f32_bits(pad), SKEL_AXIS_ROW, in, out, false);
}

skel_status skel_mapoverlap_1d_matrix(skel_ctx* c, const float* w, int r, skel_edge edge, double pad, skel_axis axis,
                                      const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap1d_impl(c, SKEL_F32, w, r, edge, f32_bits(pad), axis, in, out, true);
}

skel_status skel_mapoverlap_2d(skel_ctx* c, const float* W, int ry, int rx, skel_edge edge, double pad,
                               const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap2d_impl(c, SKEL_F32, W, ry, rx, edge, f32_bits(pad), in, out);
}

skel_status skel_mapoverlap_1d_i32(skel_ctx* c, const int32_t* w, int r, skel_edge edge, int32_t pad,
                                   const skel_vector* in, skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap1d_impl(c, SKEL_I32, w, r, edge, static_cast<uint32_t>(pad), SKEL_AXIS_ROW, in, out, false);
}

skel_status skel_mapoverlap_1d_matrix_i32(skel_ctx* c, const int32_t* w, int r, skel_edge edge, int32_t pad, skel_axis axis,
                                          const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap1d_impl(c, SKEL_I32, w, r, edge, static_cast<uint32_t>(pad), axis, in, out, true);
}

skel_status skel_mapoverlap_2d_i32(skel_ctx* c, const int32_t* W, int ry, int rx, skel_edge edge, int32_t pad,
                                   const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap2d_impl(c, SKEL_I32, W, ry, rx, edge, static_cast<uint32_t>(pad), in, out);
}

skel_status skel_mapoverlap_1d_f64(skel_ctx* c, const double* w, int r, skel_edge edge, double pad, const skel_vector* in,
                                   skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap_f64_impl(c, SKEL_SK_OVERLAP1D, w, r, 0, edge, pad, in, out, false);
}

skel_status skel_mapoverlap_1d_matrix_f64(skel_ctx* c, const double* w, int r, skel_edge edge, double pad, skel_axis axis,
                                          const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  if (axis != SKEL_AXIS_ROW && axis != SKEL_AXIS_COL) return fail(c, SKEL_ERR_INVALID_ARG, "bad axis");
  return overlap_f64_impl(c, axis == SKEL_AXIS_ROW ? SKEL_SK_OVERLAP1D : SKEL_SK_OVERLAP1D_COL, w, r, 0, edge, pad, in, out, true);
}

skel_status skel_mapoverlap_2d_f64(skel_ctx* c, const double* W, int ry, int rx, skel_edge edge, double pad,
                                   const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle");
  return overlap_f64_impl(c, SKEL_SK_OVERLAP2D, W, ry, rx, edge, pad, in, out, true);
}

skel_status skel_mapoverlap_separable(skel_ctx* c, const float* w_row, int r_row, const float* w_col, int r_col,
                                      skel_edge edge, double pad, const skel_matrix* in, skel_matrix* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!mat_ok(in) || !mat_ok(out) || !w_row || !w_col) return fail(c, SKEL_ERR_INVALID_ARG, "bad handle or NULL weights");
  if (r_row < 0 || r_col < 0 || r_row > SKEL_MAX_RADIUS_1D || r_col > SKEL_MAX_RADIUS_1D)
    return fail(c, SKEL_ERR_UNSUPPORTED, "radius out of range");
  skel_status st = overlap_check(c, in, out, edge);
  if (st != SKEL_OK) return st;
  Call k;
  k.inst.skeleton = SKEL_SK_SEPARABLE;
  k.inst.fn = SKEL_FN_WSTENCIL;
  k.inst.dtype = SKEL_F32;
  k.inst.r0 = r_row;
  k.inst.r1 = r_col;
  k.inst.edge = edge;
  k.pad = static_cast<float>(pad);
  memcpy(k.w1.w, w_row, sizeof(float) * (2 * r_row + 1));
  memcpy(k.w1b.w, w_col, sizeof(float) * (2 * r_col + 1));
  k.rows = in->rows;
  k.cols = in->cols;
  return overlap_run(c, k, in, out);
}

// ---- Scan -------------------------------------------------------------------------------------------
skel_status skel_scan(skel_ctx* c, skel_fn op, skel_scan_mode mode, double init, const skel_vector* in, skel_vector* out) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (!vec_ok(in) || !vec_ok(out)) return fail(c, SKEL_ERR_INVALID_ARG, "bad vector handle");
  if (!red_op_ok(op)) return fail(c, SKEL_ERR_UNSUPPORTED, "scan operator must be ADD, MULT or MAX");
  if (mode != SKEL_SCAN_INCLUSIVE && mode != SKEL_SCAN_EXCLUSIVE) return fail(c, SKEL_ERR_INVALID_ARG, "bad scan mode");
  Storage* a = in->st;
  Storage* o = out->st;
  if (a->dtype != o->dtype) return fail(c, SKEL_ERR_DTYPE, "operand element types differ");
  if (a->n != o->n) return fail(c, SKEL_ERR_SIZE_MISMATCH, "operand sizes differ");
  Call k;
  k.inst.skeleton = SKEL_SK_SCAN;
  k.inst.fn = op;
  k.inst.dtype = a->dtype;
  k.inst.mode = mode;
  k.c64 = mode == SKEL_SCAN_EXCLUSIVE ? init : 0.0;
  skel_status st = const_bits(c, a->dtype, mode == SKEL_SCAN_EXCLUSIVE ? init : 0.0, &k.cbits);
  if (st != SKEL_OK) return st;
  OperandSet set;
  set.add(a, ACC_READ);
  set.add(o, ACC_WRITE);
  st = acquire_all(c, set);
  if (st != SKEL_OK) return st;
  k.in0 = a->dev;
  k.out = o->dev;
  k.n = a->n;
  if (k.n > 0) {
    st = run_call(c, k);
    if (st != SKEL_OK) return st;
  }
  return publish_all(c, set);
}

// ---- selector ---------------------------------------------------------------------------------------
int skel_variant_count(int skeleton) { return variant_count(skeleton); }
const char* skel_variant_name(int skeleton, int variant) { return variant_name(skeleton, variant); }

skel_status skel_plan_save(skel_ctx* c, const char* path) {
  if (!ctx_ok(c) || !path) return SKEL_ERR_INVALID_ARG;
  return c->plan.save(path) ? SKEL_OK : fail(c, SKEL_ERR_IO, "cannot write plan file");
}

skel_status skel_plan_load(skel_ctx* c, const char* path) {
  if (!ctx_ok(c) || !path) return SKEL_ERR_INVALID_ARG;
  return c->plan.load(path) ? SKEL_OK : fail(c, SKEL_ERR_IO, "cannot read or parse plan file");
}

skel_status skel_plan_clear(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  c->plan.clear();
  return SKEL_OK;
}

skel_status skel_plan_lookup(skel_ctx* c, const skel_instance* inst, size_t n, int* variant) {
  if (!ctx_ok(c) || !inst || !variant) return SKEL_ERR_INVALID_ARG;
  if (inst->skeleton < 0 || inst->skeleton >= SKEL_SK_COUNT) return fail(c, SKEL_ERR_INVALID_ARG, "bad skeleton id");
  int v = c->forced[inst->skeleton];
  if (v < 0) v = c->plan.lookup(key_of(*inst), n);
  if (v < 0 || v >= variant_count(inst->skeleton)) {
    int cnt = 0;
    const int* pref = preference(inst->skeleton, inst->dtype, &cnt);
    v = cnt > 0 ? pref[0] : -1;
  }
  *variant = v;
  return SKEL_OK;
}

skel_status skel_plan_explain(skel_ctx* c, const skel_instance* inst, size_t n, int* variant, int* exact,
                              int* variant_from_plan) {
  if (!ctx_ok(c) || !inst || !variant || !exact || !variant_from_plan) return SKEL_ERR_INVALID_ARG;
  if (inst->skeleton < 0 || inst->skeleton >= SKEL_SK_COUNT) return fail(c, SKEL_ERR_INVALID_ARG, "bad skeleton id");
  bool ex = false;
  int v = c->plan.lookup(key_of(*inst), n, &ex);
  *exact = ex ? 1 : 0;
  *variant_from_plan = (v >= 0 && v < variant_count(inst->skeleton)) ? 1 : 0;
  if (!*variant_from_plan) {
    int cnt = 0;
    const int* pref = preference(inst->skeleton, inst->dtype, &cnt);
    v = cnt > 0 ? pref[0] : -1;
    *exact = 0;
  }
  *variant = v;
  return SKEL_OK;
}

skel_status skel_plan_set(skel_ctx* c, const skel_instance* inst, size_t n_min, int variant) {
  if (!ctx_ok(c) || !inst) return SKEL_ERR_INVALID_ARG;
  if (inst->skeleton < 0 || inst->skeleton >= SKEL_SK_COUNT) return fail(c, SKEL_ERR_INVALID_ARG, "bad skeleton id");
  if (variant < 0 || variant >= variant_count(inst->skeleton)) return fail(c, SKEL_ERR_INVALID_ARG, "bad variant id");
  c->plan.set(key_of(*inst), n_min, variant);
  return SKEL_OK;
}

skel_status skel_force_variant(skel_ctx* c, int skeleton, int variant) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (skeleton < 0 || skeleton >= SKEL_SK_COUNT) return fail(c, SKEL_ERR_INVALID_ARG, "bad skeleton id");
  if (variant < -1 || variant >= variant_count(skeleton)) return fail(c, SKEL_ERR_INVALID_ARG, "bad variant id");
  c->forced[skeleton] = variant;
  return SKEL_OK;
}

skel_status skel_last_variant(skel_ctx* c, int* skeleton, int* variant) {
  if (!ctx_ok(c) || !skeleton || !variant) return SKEL_ERR_INVALID_ARG;
  *skeleton = c->last_sk;
  *variant = c->last_var;
  return SKEL_OK;
}

skel_status skel_tune_table(skel_ctx* c, float* times_us, size_t capacity, size_t* count) {
  if (!ctx_ok(c) || !count) return SKEL_ERR_INVALID_ARG;
  *count = c->tune_table.size();
  if (times_us) memcpy(times_us, c->tune_table.data(), sizeof(float) * std::min(capacity, c->tune_table.size()));
  return SKEL_OK;
}

namespace {
// device buffers and events of one tuning run, released on every exit path
struct TuneResources {
  void* arena[3] = {nullptr, nullptr, nullptr};  // operand 0, operand 1, output: each holds `slots` rotating buffers
  void* dirty = nullptr;                          // the writer's target: larger than the L2 cache
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  ~TuneResources() {
    for (void* a : arena)
      if (a) cudaFree(a);
    if (dirty) cudaFree(dirty);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
  }
};
}  // namespace

skel_status skel_tune_instance(skel_ctx* c, const skel_instance* inst, int log2_lo, int log2_hi, size_t cols, int reps) {
  if (!ctx_ok(c) || !inst) return SKEL_ERR_INVALID_ARG;
  const int sk = inst->skeleton;
  if (sk < 0 || sk >= SKEL_SK_COUNT) return fail(c, SKEL_ERR_INVALID_ARG, "bad skeleton id");
  if (log2_lo < 0 || log2_hi > 32 || log2_lo > log2_hi || reps < 1) return fail(c, SKEL_ERR_INVALID_ARG, "bad tuning range");
  if (inst->dtype == SKEL_F64) return fail(c, SKEL_ERR_UNSUPPORTED, "fp64 elements have one kernel per skeleton: nothing to tune");
  const bool matrix = sk == SKEL_SK_OVERLAP1D_COL || sk == SKEL_SK_OVERLAP2D || sk == SKEL_SK_SEPARABLE ||
                      sk == SKEL_SK_REDUCE_ROWS ||
                      (sk == SKEL_SK_OVERLAP1D && cols > 0);
  if (matrix && cols == 0) return fail(c, SKEL_ERR_INVALID_ARG, "matrix skeletons need cols");
  skel_status st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  const size_t nmax = size_t(1) << log2_hi;
  st = ensure_scan_state(c, nmax);
  if (st != SKEL_OK) return st;
  // Conditions of a sustained run (the ones bench.py times under): every launch takes its operands from the next
  // slot of an arena of at least ARENA_MIN bytes (> 2 x the 126 MB L2: no launch finds its input in the cache),
  // and is preceded by a writer that leaves the L2 full of dirty lines, like the skeleton call before it in a
  // real sequence. A tuner that re-reads one buffer ranks near-equal variants differently from the bench.
  constexpr size_t ARENA_MIN = size_t(384) << 20, DIRTY_BYTES = size_t(160) << 20;
  const size_t arena_bytes = std::max(nmax * 4, ARENA_MIN);
  TuneResources R;
  for (void*& a : R.arena) CU(c, cudaMalloc(&a, arena_bytes));
  CU(c, cudaMalloc(&R.dirty, DIRTY_BYTES));
  {
    // Pseudo-random operands, not zeros: an all-zero stream draws less HBM power than real data, and a
    // plan tuned on it picks variants that lose under the power cap of a sustained run. The bit
    // patterns are floats in [1, 2) (as int32 they are large values that wrap in sums: harmless).
    const size_t total = arena_bytes / 4;
    const size_t chunk = std::min<size_t>(total, size_t(1) << 22);
    std::vector<uint32_t> host(chunk);
    uint64_t z = 0x9E3779B97F4A7C15ull;
    for (size_t i = 0; i < chunk; ++i) {
      z ^= z << 13;
      z ^= z >> 7;
      z ^= z << 17;
      host[i] = 0x3F800000u | static_cast<uint32_t>(z >> 41);
    }
    for (void* b : R.arena) {
      CU(c, cudaMemcpyAsync(b, host.data(), chunk * 4, cudaMemcpyHostToDevice, c->stream));
      for (size_t done = chunk; done < total; done *= 2)  // double the filled prefix
        CU(c, cudaMemcpyAsync(static_cast<char*>(b) + done * 4, b, std::min(done, total - done) * 4,
                              cudaMemcpyDeviceToDevice, c->stream));
    }
    CU(c, cudaStreamSynchronize(c->stream));
  }
  CU(c, cudaEventCreate(&R.e0));
  CU(c, cudaEventCreate(&R.e1));
  const int nv = variant_count(sk);
  c->tune_table.assign(size_t(log2_hi - log2_lo + 1) * nv, std::numeric_limits<float>::quiet_NaN());
  const InstanceKey key = key_of(*inst);
  bool erased = false;  // the old entry goes when the first size has been timed successfully
  int prev_best = -1;
  size_t prev_n = 0;
  skel_status result = SKEL_OK;
  size_t rot = 0;  // rotating slot counter
  auto make_call = [&](size_t n, Call& k) -> bool {  // false: size not representable (matrix smaller than a row)
    k.inst = *inst;
    k.n = n;
    k.rows = 1;
    k.cols = n;
    if (matrix) {
      if (n < cols) return false;
      k.cols = cols;
      k.rows = n / cols;
      k.n = k.rows * cols;
    }
    for (int i = 0; i < 129; ++i) k.w1.w[i] = k.w1b.w[i] = 1.0f / 129.0f;
    for (int i = 0; i < 17 * 17; ++i) k.w2.w[i] = 1.0f / 289.0f;
    return true;
  };
  auto point_at_slot = [&](Call& k) {  // operands of the next launch: the next slot of each arena
    const size_t slot_bytes = (k.n * 4 + 1023) / 1024 * 1024;  // keeps every alignment the variants ask for
    const size_t slots = std::max<size_t>(1, std::min<size_t>(arena_bytes / std::max<size_t>(slot_bytes, 1), 256));
    const size_t off = (rot++ % slots) * slot_bytes;
    char* a0 = static_cast<char*>(R.arena[0]) + off;
    char* a1 = static_cast<char*>(R.arena[1]) + off;
    char* a2 = static_cast<char*>(R.arena[2]) + off;
    k.in0 = a0;
    k.in1 = (sk == SKEL_SK_MAP || sk == SKEL_SK_MAPREDUCE) && inst->mode ? a1 : nullptr;
    k.in2 = (sk == SKEL_SK_MAP && inst->fn == SKEL_FN_MULADD) ? a0 : nullptr;
    k.out = (sk == SKEL_SK_REDUCE || sk == SKEL_SK_MAPREDUCE) ? c->d_result : static_cast<void*>(a2);
  };
  // Mean of the middle half of `reps` launches (the lowest and the highest quarter are dropped) of every variant in
  // `vs`, INTERLEAVED (rep-major): clock and power state drift during a tuning run (sw_power_cap), and timing one
  // variant after the other mis-ranks near-equal ones. Not the median: CUDA event timestamps tick in steps of about
  // 2 us on this driver, so a median of single launches is quantised to that step (4 % of a 47 us Reduce, more than
  // the differences the plan is about), while the phase of a launch against the tick is random and a mean resolves it.
  std::vector<std::vector<float>> tsamp;
  auto time_variants = [&](Call k, const std::vector<int>& vs, std::vector<float>& med_us) -> bool {
    tsamp.assign(vs.size(), std::vector<float>());
    for (int rep = -1; rep < reps; ++rep) {  // rep -1 is the warm-up
      for (size_t j = 0; j < vs.size(); ++j) {
        point_at_slot(k);
        if (cudaMemsetAsync(R.dirty, rep & 0xff, DIRTY_BYTES, c->stream) != cudaSuccess) return false;  // dirty L2
        cudaEventRecord(R.e0, c->stream);
        const bool bad = launch_call(c, k, vs[j]) != cudaSuccess;
        cudaEventRecord(R.e1, c->stream);
        if (cudaEventSynchronize(R.e1) != cudaSuccess || bad) return false;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, R.e0, R.e1);
        if (rep >= 0) tsamp[j].push_back(ms * 1000.f);
      }
    }
    med_us.resize(vs.size());
    for (size_t j = 0; j < vs.size(); ++j) {
      std::sort(tsamp[j].begin(), tsamp[j].end());
      const int lo = reps / 4, hi = reps - reps / 4;
      float sum = 0.f;
      for (int r = lo; r < hi; ++r) sum += tsamp[j][r];
      med_us[j] = sum / float(hi - lo);
    }
    return true;
  };
  std::vector<int> vs;
  std::vector<float> meds;
  for (int lg = log2_lo; lg <= log2_hi && result == SKEL_OK; ++lg) {
    Call k;
    if (!make_call(size_t(1) << lg, k)) continue;
    point_at_slot(k);
    float best_t = 0.f;
    int best = -1;
    vs.clear();
    for (int v = 0; v < nv; ++v)
      if (variant_ok(k, v)) vs.push_back(v);
    if (!time_variants(k, vs, meds)) {
      result = cuda_fail(c, cudaGetLastError(), "tuning launch");
      break;
    }
    if (!erased) {
      c->plan.erase(key);
      erased = true;
    }
    for (size_t j = 0; j < vs.size(); ++j) {
      c->tune_table[size_t(lg - log2_lo) * nv + vs[j]] = meds[j];
      if (best < 0 || meds[j] < best_t) {  // ties -> lower variant id
        best = vs[j];
        best_t = meds[j];
      }
    }
    // hysteresis: keep the previous size's winner unless it is more than 1.5 % AND more than 0.5 us slower than
    // the best here (timing noise otherwise turns the plan into a list of spurious breakpoints, above all at
    // the launch-latency-bound small sizes where every variant takes the same few microseconds)
    if (best >= 0 && prev_best >= 0 && prev_best != best) {
      const float tp = c->tune_table[size_t(lg - log2_lo) * nv + prev_best];
      if (tp == tp && (tp <= 1.015f * best_t || tp <= best_t + 0.5f)) best = prev_best;
    }
    if (best >= 0 && best != prev_best) {
      size_t n_min = prev_best < 0 ? 0 : k.n;
      if (prev_best >= 0) {
        // Adaptive refinement (adaptive sampling of the context space): the winner changes
        // somewhere in (prev_n, k.n]; bisect that interval (geometric midpoints, rounded to whole rows / 1024
        // elements), timing only the two contenders, until it is narrower than 2^(1/4).
        size_t lo = prev_n, hi = k.n;
        const size_t gran = matrix ? cols : 1024;
        while (result == SKEL_OK && double(hi) / double(lo) > 1.19) {
          size_t mid = static_cast<size_t>(std::sqrt(double(lo) * double(hi))) / gran * gran;
          if (mid <= lo || mid >= hi) break;
          Call m;
          if (!make_call(mid, m)) break;
          point_at_slot(m);
          if (!variant_ok(m, prev_best) || !variant_ok(m, best)) break;
          if (!time_variants(m, {prev_best, best}, meds)) {
            result = cuda_fail(c, cudaGetLastError(), "tuning launch");
            break;
          }
          const float t_old = meds[0], t_new = meds[1];
          if (t_old <= 1.015f * t_new || t_old <= t_new + 0.5f) lo = mid;  // the old winner still holds (same hysteresis)
          else hi = mid;
        }
        n_min = hi;
      }
      c->plan.set(key, n_min, best);
      prev_best = best;
    }
    prev_n = k.n;
    c->stats.launches += c->launches;
    c->launches = 0;
  }
  return result;
}

// ---- container-layer overhead measurement (skel.h skel_replay_*) ------------------------------------------
skel_status skel_replay_begin(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  if (c->fusion) return fail(c, SKEL_ERR_UNSUPPORTED, "recording needs cross-call fusion off");
  skel_status st = flush_pending(c);
  if (st != SKEL_OK) return st;
  c->recorded.clear();
  c->recording = true;
  return SKEL_OK;
}

skel_status skel_replay_end(skel_ctx* c, int* ncalls) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  c->recording = false;
  while (!c->recorded.empty() && c->recorded.back().variant == -1000) c->recorded.pop_back();  // a call that failed
  if (ncalls) *ncalls = static_cast<int>(c->recorded.size());
  return SKEL_OK;
}

skel_status skel_replay_run(skel_ctx* c, int raw, int reps, double* host_us, double* dev_us) {
  if (!ctx_ok(c) || !host_us || !dev_us || reps < 1) return SKEL_ERR_INVALID_ARG;
  if (c->recording) return fail(c, SKEL_ERR_BUSY, "still recording: call skel_replay_end first");
  if (c->recorded.empty()) return fail(c, SKEL_ERR_INVALID_ARG, "nothing recorded");
  if (c->fusion) return fail(c, SKEL_ERR_UNSUPPORTED, "replay needs cross-call fusion off");
  skel_status st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  CU(c, cudaStreamSynchronize(c->stream));
  cudaEvent_t e0, e1;
  CU(c, cudaEventCreate(&e0));
  CU(c, cudaEventCreate(&e1));
  skel_status result = SKEL_OK;
  timespec t0, t1;
  clock_gettime(CLOCK_MONOTONIC, &t0);
  cudaEventRecord(e0, c->stream);
  for (int rep = 0; rep < reps && result == SKEL_OK; ++rep) {
    for (RecordedCall& r : c->recorded) {
      if (raw) {
        if (r.k.inst.skeleton == SKEL_SK_SCAN)
          result = r.k.inst.dtype == SKEL_F64 ? ensure_scan_state64(c, r.k.n) : ensure_scan_state(c, r.k.n);
        if (result == SKEL_OK && (r.k.inst.dtype == SKEL_F64 ? launch_call_f64(c, r.k) : launch_call(c, r.k, r.variant)) != cudaSuccess)
          result = cuda_fail(c, cudaGetLastError(), "replay launch");
        c->stats.launches += c->launches;
        c->launches = 0;
      } else {
        OperandSet set = r.set;
        result = acquire_all(c, set);
        if (result == SKEL_OK) result = run_call(c, r.k);
        if (result == SKEL_OK) result = publish_all(c, set);
      }
      if (result != SKEL_OK) break;
    }
  }
  cudaEventRecord(e1, c->stream);
  clock_gettime(CLOCK_MONOTONIC, &t1);  // enqueue time: the calls are asynchronous
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (result != SKEL_OK) return result;
  if (e != cudaSuccess) return cuda_fail(c, e, "replay");
  *host_us = ((t1.tv_sec - t0.tv_sec) * 1e9 + (t1.tv_nsec - t0.tv_nsec)) / 1e3 / reps;
  *dev_us = double(ms) * 1e3 / reps;
  return SKEL_OK;
}

// ---- observability ------------------------------------------------------------------------------------
skel_status skel_get_stats(skel_ctx* c, skel_stats* out) {
  if (!ctx_ok(c) || !out) return SKEL_ERR_INVALID_ARG;
  *out = c->stats;
  return SKEL_OK;
}

skel_status skel_probe_fma_with_loads(skel_ctx* c, int nl, int reps, double* fma_per_s) {
  if (!ctx_ok(c) || !fma_per_s || reps < 1) return SKEL_ERR_INVALID_ARG;
  if (nl != 0 && nl != 1 && nl != 2 && nl != 4 && nl != 8) return fail(c, SKEL_ERR_INVALID_ARG, "lds128_per_iter must be 0, 1, 2, 4 or 8");
  skel_status st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  cudaEvent_t e0, e1;
  CU(c, cudaEventCreate(&e0));
  CU(c, cudaEventCreate(&e1));
  Launch L{c->stream, c->sms, &c->launches, c->tile_ctr, &c->tile_next};
  std::vector<float> ms(reps);
  double count = 0;
  cudaError_t e = cudaSuccess;
  const float* in64 = static_cast<const float*>(c->scratch.partials);  // any 64 readable floats
  for (int r = -1; r < reps && e == cudaSuccess; ++r) {  // r = -1 warms up
    cudaEventRecord(e0, c->stream);
    e = launch_fma_lds_probe(L, nl, in64, static_cast<float*>(c->d_result), &count);
    cudaEventRecord(e1, c->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float t = 0.f;
    if (e == cudaSuccess) cudaEventElapsedTime(&t, e0, e1);
    if (r >= 0) ms[r] = t;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  c->stats.launches += c->launches;
  c->launches = 0;
  if (e != cudaSuccess) return cuda_fail(c, e, "FMA + LDS probe");
  std::sort(ms.begin(), ms.end());
  *fma_per_s = count / (double(ms[reps / 2]) * 1e-3);
  return SKEL_OK;
}

skel_status skel_probe_fma_peak(skel_ctx* c, int reps, double* fma_per_s) {
  if (!ctx_ok(c) || !fma_per_s || reps < 1) return SKEL_ERR_INVALID_ARG;
  skel_status st = ensure_device(c);
  if (st != SKEL_OK) return st;
  st = flush_pending(c);
  if (st != SKEL_OK) return st;
  cudaEvent_t e0, e1;
  CU(c, cudaEventCreate(&e0));
  CU(c, cudaEventCreate(&e1));
  Launch L{c->stream, c->sms, &c->launches, c->tile_ctr, &c->tile_next};
  std::vector<float> ms(reps);
  double count = 0;
  for (int r = -1; r < reps; ++r) {  // r = -1 warms up
    cudaEventRecord(e0, c->stream);
    cudaError_t e = launch_fma_probe(L, static_cast<float*>(c->d_result), &count);
    cudaEventRecord(e1, c->stream);
    if (e != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) {
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      return cuda_fail(c, e != cudaSuccess ? e : cudaGetLastError(), "FMA probe");
    }
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    if (r >= 0) ms[r] = t;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  std::sort(ms.begin(), ms.end());
  *fma_per_s = count / (double(ms[reps / 2]) * 1e-3);
  c->stats.launches += c->launches;
  c->launches = 0;
  return SKEL_OK;
}

skel_status skel_reset_stats(skel_ctx* c) {
  if (!ctx_ok(c)) return SKEL_ERR_INVALID_ARG;
  c->stats = skel_stats{};
  return SKEL_OK;
}

skel_status skel_ranges_add(uint64_t* ranges, size_t* count, size_t capacity, uint64_t begin, uint64_t end) {
  if (!ranges || !count || *count >= capacity) return SKEL_ERR_INVALID_ARG;
  static_assert(sizeof(ElemRange) == 2 * sizeof(uint64_t), "pairs of 64-bit bounds");
  *count = ranges_add(reinterpret_cast<ElemRange*>(ranges), *count, begin, end);
  return SKEL_OK;
}

skel_status skel_coherence_step(int state, int actor, skel_access access, skel_coherence mode, int* new_state, int* transfer) {
  if (state < 0 || state > 3 || (actor != 0 && actor != 1) || access < 0 || access > 2 || (mode != SKEL_LAZY && mode != SKEL_EAGER) ||
      !new_state || !transfer)
    return SKEL_ERR_INVALID_ARG;
  const CoherenceStep s = coherence_step(state, actor, access, mode);
  *new_state = s.new_state;
  *transfer = s.transfer;
  return s.ok ? SKEL_OK : SKEL_ERR_UNINIT;
}

}  // extern "C"
#pragma GCC visibility pop
