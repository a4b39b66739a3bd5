// Scan skeleton (PAPER.md L75/L83 name it; definition: DESIGN.md reading 4):
//   inclusive out[i] = x[0] (+) ... (+) x[i];  exclusive out[0] = init, out[i] = init (+) x[0..i-1].
//
// Variants:
//  * "lookback_*": single pass, 8 B/elem. Tiles are handed out by an atomic ticket (forward
//    progress does not depend on block scheduling order); a tile publishes (epoch|status|value) as
//    ONE 64-bit word, so no fence is needed between status and value; its warp 0 looks back over
//    windows of 32 predecessors. The epoch tag makes a memset of the tile states between calls
//    unnecessary. i32 only: with floating point the result would depend on how far each look-back
//    happened to reach.
//  * "persist_*": the same with a grid of co-resident blocks walking strided tiles (no ticket).
//  * "ws_*": warp-specialised persistent CTAs fed by a shared-memory ring of bulk async copies;
//    one prefix warp per stage publishes the aggregate as soon as the tile lands.
//  * "l2ahead_*": the fastest at large n (6.2 TB/s at 2^28): a TMA-fed reduce pass runs D tiles
//    ahead and publishes aggregates, a prefix warp sums them (no chain), the scan pass re-reads the
//    tile from L2. See the comment above scan_l2_kernel.
//  * "three_kernel_*": reduce per block -> scan of the block sums -> rescan with carry. 12 B/elem,
//    fixed combination order (deterministic for f32); the correctness anchor for the look-back.
#include "common.cuh"
#include "kernels.hpp"
#include <stdlib.h>

namespace skel {
namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int LB_WINDOWS = 1;  // look-back windows (of 32 tile states) fetched per round

template <typename T, int OP> __device__ __forceinline__ T op2(T a, T b) { return apply_fn<OP>(T(0), a, b); }

// Scan state shared by the two phases of one tile (registers + the tile's aggregate).
template <typename T, int V, int U> struct TileRegs {
  T x[U][V];       // phase A: inclusive scan inside each V-vector
  T lane_excl[U];  // exclusive prefix of this thread's vector u inside its warp
};

// Phase A: load the tile, scan locally, return the tile aggregate (all threads).
// smem layout: tot[E] | excl[E] | agg, E = U * (THREADS/32).
template <typename T, int OP, int THREADS, int V, int U, bool NC>
__device__ __forceinline__ T tile_phase_a(const T* in, size_t base, size_t n, TileRegs<T, V, U>& R, T* sm,
                                          const T* staged = nullptr) {
  constexpr int NW = THREADS / 32, E = U * NW, EPL = (E + 31) / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const T ident = identity<T, OP>();
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const size_t i0 = base + (size_t(u) * THREADS + threadIdx.x) * V;
    if (staged != nullptr) {  // the whole tile was staged in shared memory by a bulk copy
      static_assert(V == 4 || V == 1 || V == 8 || V == 2, "vector width");
      if constexpr (V == 4) {
        const uint4 q = *reinterpret_cast<const uint4*>(staged + (u * THREADS + threadIdx.x) * 4);
        R.x[u][0] = from_bits<T>(q.x); R.x[u][1] = from_bits<T>(q.y);
        R.x[u][2] = from_bits<T>(q.z); R.x[u][3] = from_bits<T>(q.w);
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j) R.x[u][j] = staged[(u * THREADS + threadIdx.x) * V + j];
      }
    } else if (i0 + V <= n) {
      uint32_t raw[V];
      ld_stream<V, NC>(raw, in + i0);
#pragma unroll
      for (int j = 0; j < V; ++j) R.x[u][j] = from_bits<T>(raw[j]);
    } else {
#pragma unroll
      for (int j = 0; j < V; ++j) R.x[u][j] = (i0 + j < n) ? in[i0 + j] : ident;
    }
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
#pragma unroll
    for (int j = 1; j < V; ++j) R.x[u][j] = op2<T, OP>(R.x[u][j - 1], R.x[u][j]);
    T ws = R.x[u][V - 1];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T y = __shfl_up_sync(FULL, ws, o);
      if (lane >= o) ws = op2<T, OP>(y, ws);
    }
    T ex = __shfl_up_sync(FULL, ws, 1);
    R.lane_excl[u] = lane == 0 ? ident : ex;
    if (lane == 31) sm[u * NW + warp] = ws;
  }
  __syncthreads();
  if (warp == 0) {
    T v[EPL];
    T run = ident;
#pragma unroll
    for (int k = 0; k < EPL; ++k) {
      const int e = lane * EPL + k;
      v[k] = e < E ? sm[e] : ident;
      run = op2<T, OP>(run, v[k]);
    }
    T ws = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T y = __shfl_up_sync(FULL, ws, o);
      if (lane >= o) ws = op2<T, OP>(y, ws);
    }
    T ex = __shfl_up_sync(FULL, ws, 1);
    ex = lane == 0 ? ident : ex;
#pragma unroll
    for (int k = 0; k < EPL; ++k) {
      const int e = lane * EPL + k;
      if (e < E) sm[E + e] = ex;
      ex = op2<T, OP>(ex, v[k]);
    }
    if (lane == 31) sm[2 * E] = ws;
  }
  __syncthreads();
  return sm[2 * E];
}

// Phase B: write the outputs given the tile's exclusive prefix `carry`.
template <typename T, int OP, int THREADS, int V, int U>
__device__ __forceinline__ void tile_phase_b(T* out, size_t base, size_t n, const TileRegs<T, V, U>& R, const T* sm,
                                             T carry, bool exclusive) {
  constexpr int NW = THREADS / 32, E = U * NW;
  const int warp = threadIdx.x >> 5;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const T p = op2<T, OP>(op2<T, OP>(carry, sm[E + u * NW + warp]), R.lane_excl[u]);
    T o[V];
#pragma unroll
    for (int j = 0; j < V; ++j) {
      if (exclusive) o[j] = j == 0 ? p : op2<T, OP>(p, R.x[u][j - 1]);
      else o[j] = op2<T, OP>(p, R.x[u][j]);
    }
    const size_t i0 = base + (size_t(u) * THREADS + threadIdx.x) * V;
    if (i0 + V <= n) {
      uint32_t raw[V];
#pragma unroll
      for (int j = 0; j < V; ++j) raw[j] = to_bits(o[j]);
      st_stream<V>(out + i0, raw);
    } else {
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (i0 + j < n) out[i0 + j] = o[j];
    }
  }
}

// ---- single pass, decoupled look-back ----------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long pack_state(uint32_t epoch, unsigned status, uint32_t value) {
  return (static_cast<unsigned long long>(epoch) << 34) | (static_cast<unsigned long long>(status) << 32) | value;
}

// Look-back of one tile, executed by warp 0 (all 32 lanes). Publishes the tile's aggregate, folds
// the predecessors' aggregates back to the nearest inclusive prefix, publishes the tile's inclusive
// prefix and returns the tile's exclusive prefix (carry).

template <typename T, int OP, int K = LB_WINDOWS>
__device__ __forceinline__ T lookback_warp0(unsigned long long* state, uint32_t epoch, unsigned tile, T agg, T init,
                                            bool exclusive) {
  const int lane = threadIdx.x & 31;
  const T ident = identity<T, OP>();
  T carry;
  if (tile == 0) {
    carry = exclusive ? init : ident;
    if (lane == 0) st_state(state, pack_state(epoch, 2u, to_bits(op2<T, OP>(carry, agg))));
    return carry;
  }
  if (lane == 0) st_state(state + tile, pack_state(epoch, 1u, to_bits(agg)));
  carry = ident;
  // The inclusive-prefix frontier advances by at most one look-back window per L2 round trip, so
  // the window decides the chain speed: LB_WINDOWS * 32 predecessor states are fetched per round
  // (independent loads in flight together) and folded nearest-first.
  long long j = static_cast<long long>(tile) - 1;
  while (true) {
    unsigned long long w[K];
    unsigned st[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const long long idx = j - lane - 32 * k;
      w[k] = idx >= 0 ? ld_state(state + idx) : 0ull;
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const long long idx = j - lane - 32 * k;
      // before the first tile: a virtual inclusive prefix equal to the identity
      st[k] = idx < 0 ? 2u : ((static_cast<uint32_t>(w[k] >> 34) == epoch) ? static_cast<unsigned>(w[k] >> 32) & 3u : 0u);
    }
    int consumed = 0;
    bool done = false;
#pragma unroll
    for (int k = 0; k < K; ++k) {
      if (done || consumed != k) continue;
      if (__any_sync(FULL, st[k] == 0u)) continue;  // not published yet: poll again from this window
      const long long idx = j - lane - 32 * k;
      const T val = idx >= 0 ? from_bits<T>(static_cast<uint32_t>(w[k])) : ident;
      const unsigned incl = __ballot_sync(FULL, st[k] == 2u);
      const int first = incl ? (__ffs(incl) - 1) : 32;
      T contrib = lane <= first ? val : ident;
      contrib = warp_reduce<T, OP>(contrib);
      carry = op2<T, OP>(contrib, carry);
      consumed = k + 1;
      if (incl) done = true;
    }
    if (done) break;
    j -= 32 * consumed;
  }
  if (lane == 0) st_state(state + tile, pack_state(epoch, 2u, to_bits(op2<T, OP>(carry, agg))));
  return carry;
}

template <typename T, int OP, int THREADS, int V, int U, bool NC>
__global__ void __launch_bounds__(THREADS)
scan_lookback_kernel(const T* in, T* out, size_t n, T init, int exclusive, unsigned long long* state,
                     unsigned* ticket, uint32_t epoch, unsigned ntiles) {
  static_assert(sizeof(T) == 4, "32-bit elements");
  constexpr int NW = THREADS / 32, E = U * NW;
  constexpr size_t TILE = size_t(THREADS) * V * U;
  __shared__ T sm[2 * E + 1];
  __shared__ unsigned s_tile;
  __shared__ T s_carry;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const unsigned tile = s_tile;
  const size_t base = size_t(tile) * TILE;

  TileRegs<T, V, U> R;
  const T agg = tile_phase_a<T, OP, THREADS, V, U, NC>(in, base, n, R, sm);

  if (warp == 0) {
    const T carry = lookback_warp0<T, OP>(state, epoch, tile, agg, init, exclusive != 0);
    if (lane == 0) s_carry = carry;
  }
  __syncthreads();
  tile_phase_b<T, OP, THREADS, V, U>(out, base, n, R, sm, s_carry, exclusive != 0);
  if (threadIdx.x == 0 && tile == ntiles - 1) *ticket = 0u;  // every ticket has been drawn by now
}

// Persistent form: a grid of co-resident blocks, block b scans tiles b, b+G, b+2G, ... in that
// order (ids grow inside a block, so the smallest unfinished tile is always being worked on).
template <typename T, int OP, int THREADS, int V, int U, bool NC>
__global__ void __launch_bounds__(THREADS)
scan_lookback_persist_kernel(const T* in, T* out, size_t n, T init, int exclusive, unsigned long long* state,
                             uint32_t epoch, unsigned ntiles) {
  constexpr int NW = THREADS / 32, E = U * NW;
  constexpr size_t TILE = size_t(THREADS) * V * U;
  __shared__ T sm[2 * E + 1];
  __shared__ T s_carry;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (unsigned tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t base = size_t(tile) * TILE;
    TileRegs<T, V, U> R;
    const T agg = tile_phase_a<T, OP, THREADS, V, U, NC>(in, base, n, R, sm);
    if (warp == 0) {
      const T carry = lookback_warp0<T, OP>(state, epoch, tile, agg, init, exclusive != 0);
      if (lane == 0) s_carry = carry;
    }
    __syncthreads();
    tile_phase_b<T, OP, THREADS, V, U>(out, base, n, R, sm, s_carry, exclusive != 0);
    __syncthreads();
  }
}

// ---- single pass, warp-specialised persistent CTAs ("ws") ------------------------------------------
// Measured on B200: in the one-tile-per-block kernel a tile spends
// ~2/3 of its life spinning in the look-back, not because the chain is long but because the load
// latency under a saturated HBM has a heavy tail (p50 2.5 us, p99 7 us) and a tile's aggregate is
// only published once ITS loads have landed; every later tile waits for the slowest earlier one,
// and while it waits its registers hold no loads in flight. The same kernel without the look-back
// runs at copy speed. This kernel takes the look-back off the data path:
//  * CTA b owns tiles b, b+G, b+2G, ... (static; cooperative launch => all CTAs co-resident).
//  * A ring of S shared-memory stages per CTA is filled by bulk async copies (TMA engine), so up to
//    S tiles per SM are in flight or waiting no matter what the look-back does.
//  * Stage s has its own PREFIX WARP: as soon as the tile lands it sums the NSW sub-tiles, publishes
//    the tile aggregate (so successors never wait for more than the landing itself), runs the
//    look-back, publishes the inclusive prefix and hands carry + sub-tile prefixes to the scanners
//    through shared memory. The S prefix warps run concurrently, so one slow look-back delays
//    neither the aggregates nor the look-backs of the CTA's other staged tiles.
//  * NSW SCANNER WARPS take the stages in order; warp w scans sub-tile w (32*4*U elements) from
//    shared memory with no block-level barrier, adds carry + sub-tile prefix, and streams the
//    result to global memory with 128-bit stores; then the stage is handed back for the next copy.
// Forward progress: tile t depends only on tiles < t, which belong to co-resident CTAs at the same
// or an earlier ring position; aggregates depend on nothing but the copy.
template <typename T, int OP, int NSW, int U, int S, int K>
__global__ void __launch_bounds__((NSW + S) * 32, 1)
scan_ws_kernel(const T* in, T* out, size_t n, T init, int exclusive, unsigned long long* state, uint32_t epoch,
               unsigned ntiles) {
  static_assert(sizeof(T) == 4 && NSW <= 32, "32-bit elements");
  constexpr int SUB = 32 * 4 * U;       // elements per scanner warp and tile
  constexpr int TILE = NSW * SUB;
  constexpr unsigned TILE_BYTES = TILE * 4u;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* buf = reinterpret_cast<T*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + size_t(S) * TILE_BYTES);  // copy landed
  uint64_t* ready = full + S;                                                       // prefixes written
  uint64_t* empty = ready + S;                                                      // scanners done reading
  T* pre = reinterpret_cast<T*>(empty + S);                                         // [S][NSW] carry (+) sub-tile prefix
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned G = gridDim.x;
  const T ident = identity<T, OP>();

  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&ready[s], 1);
      mbar_init(&empty[s], NSW);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (warp >= NSW) {
    // ---------------- prefix warp of stage s ----------------
    const int s = warp - NSW;
    T* stage = buf + size_t(s) * TILE;
    unsigned use = 0;
    for (unsigned long long tile = blockIdx.x + (unsigned long long)s * G; tile < ntiles; tile += (unsigned long long)S * G, ++use) {
      const size_t base = size_t(tile) * TILE;
      const bool whole = base + TILE <= n;
      if (use > 0) mbar_wait(&empty[s], (use - 1) & 1u);
      if (whole) {
        if (lane == 0) {
          mbar_arrive_expect_tx(&full[s], TILE_BYTES);
          bulk_load(stage, in + base, TILE_BYTES, &full[s]);
        }
      } else {  // ragged last tile: guarded copy, identity padding
        for (int i = lane; i < TILE; i += 32) stage[i] = (base + i < n) ? in[base + i] : ident;
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[s]);
      }
      mbar_wait(&full[s], use & 1u);
      // sub-tile sums (same striped layout as the scanners: conflict-free 128-bit reads)
      T sub = ident;  // lane w < NSW ends up holding the sum of sub-tile w
#pragma unroll
      for (int w = 0; w < NSW; ++w) {
        T a = ident;
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const uint4 q = *reinterpret_cast<const uint4*>(stage + w * SUB + (u * 32 + lane) * 4);
          a = op2<T, OP>(a, op2<T, OP>(op2<T, OP>(from_bits<T>(q.x), from_bits<T>(q.y)),
                                       op2<T, OP>(from_bits<T>(q.z), from_bits<T>(q.w))));
        }
        a = warp_reduce<T, OP>(a);
        if (lane == w) sub = a;
      }
      // exclusive prefix of the sub-tile sums over lanes 0..NSW-1, and the tile aggregate
      T inc = sub;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        T y = __shfl_up_sync(FULL, inc, o);
        if (lane >= o) inc = op2<T, OP>(y, inc);
      }
      T exc = __shfl_up_sync(FULL, inc, 1);
      if (lane == 0) exc = ident;
      const T agg = __shfl_sync(FULL, inc, NSW - 1);
      const T carry = lookback_warp0<T, OP, K>(state, epoch, (unsigned)tile, agg, init, exclusive != 0);
      if (lane < NSW) pre[s * NSW + lane] = op2<T, OP>(carry, exc);
      __syncwarp();
      if (lane == 0) mbar_arrive(&ready[s]);
    }
  } else {
    // ---------------- scanner warp `warp`: sub-tile `warp` of every tile of this CTA ----------------
    unsigned it = 0;
    for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += G, ++it) {
      const int s = it % S;
      const unsigned use = it / S;
      const T* stage = buf + size_t(s) * TILE + warp * SUB;
      mbar_wait(&ready[s], use & 1u);
      const T p0 = pre[s * NSW + warp];
      T x[U][4];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const uint4 q = *reinterpret_cast<const uint4*>(stage + (u * 32 + lane) * 4);
        x[u][0] = from_bits<T>(q.x); x[u][1] = from_bits<T>(q.y); x[u][2] = from_bits<T>(q.z); x[u][3] = from_bits<T>(q.w);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);  // the stage may be refilled
      const size_t base = size_t(tile) * TILE + size_t(warp) * SUB;
      T run = p0;  // exclusive prefix of vector-row u of this sub-tile
#pragma unroll
      for (int u = 0; u < U; ++u) {
#pragma unroll
        for (int j = 1; j < 4; ++j) x[u][j] = op2<T, OP>(x[u][j - 1], x[u][j]);
        T ws = x[u][3];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          T y = __shfl_up_sync(FULL, ws, o);
          if (lane >= o) ws = op2<T, OP>(y, ws);
        }
        T ex = __shfl_up_sync(FULL, ws, 1);
        const T p = lane == 0 ? run : op2<T, OP>(run, ex);
        run = op2<T, OP>(run, __shfl_sync(FULL, ws, 31));
        T o4[4];
        if (exclusive) {
          o4[0] = p; o4[1] = op2<T, OP>(p, x[u][0]); o4[2] = op2<T, OP>(p, x[u][1]); o4[3] = op2<T, OP>(p, x[u][2]);
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j) o4[j] = op2<T, OP>(p, x[u][j]);
        }
        const size_t i0 = base + (size_t(u) * 32 + lane) * 4;
        if (i0 + 4 <= n) {
          uint32_t raw[4] = {to_bits(o4[0]), to_bits(o4[1]), to_bits(o4[2]), to_bits(o4[3])};
          st_stream<4>(out + i0, raw);
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (i0 + j < n) out[i0 + j] = o4[j];
        }
      }
    }
  }
}

// ---- single pass over HBM, two passes over L2 ("l2ahead") --------------------------------------------
// What bounds every chained single-pass kernel above on B200 is not the chain arithmetic but the
// load-latency tail of a saturated HBM (p50 2.5 us, p99 7 us, max ~10
// us): tile t cannot be finished before every earlier tile has LANDED, so each slot of on-chip
// buffering is held for the tail latency, not the mean, and 192 KB of shared memory per SM is not
// enough buffer. Here the buffer is the 126 MB L2 and there is no chain at all:
//  * CTA b owns tiles b, b+G, b+2G, ... (static; cooperative launch => all CTAs co-resident).
//  * REDUCE phase (worker warps): tile k+D is streamed once from HBM (loads tagged L2::evict_last),
//    summed, and its aggregate published. Order-free, never waits.
//  * PREFIX warp (one per CTA, runs ahead of the scan phase): the exclusive prefix of the CTA's
//    next tile is the prefix of its previous tile (+) the G consecutive aggregates in between - a
//    windowed sum over already-published aggregates (all loads of a window in flight together), no
//    look-back chain, no inclusive prefixes to publish. It hands the carry to the workers through a
//    small shared-memory queue.
//  * SCAN phase (worker warps): tile k is read a second time - now from L2 (evict_first, like the
//    output stores) - scanned locally, offset by the carry and streamed out.
// HBM traffic stays 8 B/elem; L2 carries 12 B/elem (+ G*8 B of aggregate reads per tile), which it
// sustains. Run-ahead = D*G tiles. Forward progress: the reduce phase
// waits for nothing; a prefix waits only for aggregates, i.e. for reduce phases.
template <int N> __device__ __forceinline__ void bar_workers() { asm volatile("bar.sync 1, %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ unsigned ld_acquire_shared(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_shared(unsigned* p, unsigned v) {
  asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

template <typename T, int OP, int NW, int U, int D, int KW, int S, int MINB>
__global__ void __launch_bounds__((NW + 1) * 32, MINB)
scan_l2_kernel(const T* in, T* out, size_t n, T init, int exclusive, unsigned long long* state, uint32_t epoch,
               unsigned ntiles) {
  static_assert(sizeof(T) == 4, "32-bit elements");
  constexpr int V = 4, WT = NW * 32, E = U * NW, Q = D + 2;
  constexpr size_t TILE = size_t(WT) * V * U;
  __shared__ T sm[2 * E + 1];
  __shared__ T red[2][NW];
  __shared__ T cq[Q];
  __shared__ unsigned cq_head, cq_tail;  // carries produced / consumed
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned long long G = gridDim.x;
  const T ident = identity<T, OP>();
  if (threadIdx.x == 0) {
    cq_head = 0;
    cq_tail = 0;
  }
  __syncthreads();

  if (warp == NW) {
    // ---------------- prefix warp ----------------
    T carry = exclusive ? init : ident;
    unsigned long long lo = 0;
    unsigned j = 0;
    for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += G, ++j) {
      // carry(tile) = carry(previous own tile) (+) aggregates of tiles [lo, tile)
      T acc = ident;
      for (unsigned long long c0 = lo; c0 < tile; c0 += 32ull * KW) {
        bool pending = true;
        unsigned long long w[KW];
        while (pending) {
          pending = false;
#pragma unroll
          for (int k = 0; k < KW; ++k) {
            const unsigned long long idx = c0 + 32ull * k + lane;
            w[k] = idx < tile ? ld_state(state + idx) : pack_state(epoch, 1u, to_bits(ident));
          }
#pragma unroll
          for (int k = 0; k < KW; ++k) pending |= static_cast<uint32_t>(w[k] >> 34) != epoch;
          pending = __any_sync(FULL, pending);
        }
#pragma unroll
        for (int k = 0; k < KW; ++k) acc = op2<T, OP>(acc, from_bits<T>(static_cast<uint32_t>(w[k])));
      }
      carry = op2<T, OP>(carry, warp_reduce<T, OP>(acc));
      lo = tile;
      while (j - ld_acquire_shared(&cq_tail) >= unsigned(Q)) {}  // queue full: wait for the workers
      if (lane == 0) {
        cq[j % Q] = carry;
        st_release_shared(&cq_head, j + 1);
      }
      __syncwarp();
    }
    return;
  }

  // ---------------- worker warps ----------------
  // The reduce pass is fed by a ring of S bulk async copies (TMA engine, L2::evict_last), so the HBM
  // stream runs S tiles ahead of the reduce, which runs D tiles ahead of the scan.
  constexpr unsigned TILE_BYTES = unsigned(TILE) * 4u;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* ring = reinterpret_cast<T*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + size_t(S) * TILE_BYTES);
  const uint64_t keep = l2_policy_evict_last(), stream = l2_policy_evict_first();
  auto red_tile = [&](unsigned j) { return blockIdx.x + (unsigned long long)j * G; };
  auto issue = [&](unsigned j) {  // thread 0: arm stage j % S with reduce-tile j (whole tiles only)
    const unsigned long long t = red_tile(j);
    if (t < ntiles && (t + 1) * TILE <= n) {
      mbar_arrive_expect_tx(&full[j % S], TILE_BYTES);
      bulk_load_hint(ring + size_t(j % S) * TILE, in + size_t(t) * TILE, TILE_BYTES, &full[j % S], keep);
    }
  };
  if (threadIdx.x == 0) {
    for (int st = 0; st < S; ++st) mbar_init(&full[st], 1);
    mbar_fence_init();
    for (unsigned j = 0; j < unsigned(S); ++j) issue(j);
  }
  bar_workers<WT>();
  unsigned par = 0;
  auto reduce_tile = [&](unsigned j) {  // sum reduce-tile j, publish its aggregate, refill its stage
    const unsigned long long tile = red_tile(j);
    const size_t base = size_t(tile) * TILE;
    T a = ident;
    if (base + TILE <= n) {
      mbar_wait(&full[j % S], (j / S) & 1u);
      const T* stage = ring + size_t(j % S) * TILE;
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const uint4 q = *reinterpret_cast<const uint4*>(stage + (u * WT + threadIdx.x) * 4);
        a = op2<T, OP>(a, op2<T, OP>(op2<T, OP>(from_bits<T>(q.x), from_bits<T>(q.y)),
                                     op2<T, OP>(from_bits<T>(q.z), from_bits<T>(q.w))));
      }
    } else {  // ragged last tile: guarded loads
      for (size_t i = base + threadIdx.x; i < n; i += WT) a = op2<T, OP>(a, in[i]);
    }
    a = warp_reduce<T, OP>(a);
    if (lane == 0) red[par][warp] = a;
    bar_workers<WT>();  // every worker has read the stage
    if (warp == 0) {
      T v = lane < NW ? red[par][lane] : ident;
      v = warp_reduce<T, OP>(v);
      if (lane == 0) {
        st_state(state + tile, pack_state(epoch, 1u, to_bits(v)));
        issue(j + S);
      }
    }
    par ^= 1u;  // red[par] is rewritten two reduces later, with worker barriers in between
  };
  auto load_tile = [&](unsigned long long tile, uint32_t (&raw)[U][V], uint64_t policy) {
    const size_t base = size_t(tile) * TILE;
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const size_t i0 = base + (size_t(u) * WT + threadIdx.x) * V;
      if (i0 + V <= n) {
        ld_hint4(raw[u], in + i0, policy);
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j) raw[u][j] = to_bits((i0 + j < n) ? in[i0 + j] : ident);
      }
    }
  };

  for (unsigned j = 0; j < unsigned(D); ++j) {  // prologue: run D tiles ahead
    if (red_tile(j) >= ntiles) break;
    reduce_tile(j);
  }
  unsigned it = 0;
  for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += G, ++it) {
    uint32_t rb[U][V];
    load_tile(tile, rb, stream);
    if (red_tile(it + D) < ntiles) reduce_tile(it + D);
    // local scan of the tile (registers)
    T x[U][V], lane_excl[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
#pragma unroll
      for (int j = 0; j < V; ++j) x[u][j] = from_bits<T>(rb[u][j]);
#pragma unroll
      for (int j = 1; j < V; ++j) x[u][j] = op2<T, OP>(x[u][j - 1], x[u][j]);
      T ws = x[u][V - 1];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        T y = __shfl_up_sync(FULL, ws, o);
        if (lane >= o) ws = op2<T, OP>(y, ws);
      }
      T ex = __shfl_up_sync(FULL, ws, 1);
      lane_excl[u] = lane == 0 ? ident : ex;
      if (lane == 31) sm[u * NW + warp] = ws;
    }
    bar_workers<WT>();
    if (warp == 0) {
      constexpr int EPL = (E + 31) / 32;
      T v[EPL];
      T run = ident;
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = lane * EPL + k;
        v[k] = e < E ? sm[e] : ident;
        run = op2<T, OP>(run, v[k]);
      }
      T ws = run;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        T y = __shfl_up_sync(FULL, ws, o);
        if (lane >= o) ws = op2<T, OP>(y, ws);
      }
      T ex = __shfl_up_sync(FULL, ws, 1);
      ex = lane == 0 ? ident : ex;
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = lane * EPL + k;
        if (e < E) sm[E + e] = ex;
        ex = op2<T, OP>(ex, v[k]);
      }
    }
    while (ld_acquire_shared(&cq_head) <= it) {}  // carry of this tile (normally long there)
    const T carry = cq[it % Q];
    bar_workers<WT>();
    const size_t base = size_t(tile) * TILE;
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const T p = op2<T, OP>(op2<T, OP>(carry, sm[E + u * NW + warp]), lane_excl[u]);
      T o[V];
#pragma unroll
      for (int j = 0; j < V; ++j) {
        if (exclusive) o[j] = j == 0 ? p : op2<T, OP>(p, x[u][j - 1]);
        else o[j] = op2<T, OP>(p, x[u][j]);
      }
      const size_t i0 = base + (size_t(u) * WT + threadIdx.x) * V;
      if (i0 + V <= n) {
        uint32_t raw[V];
#pragma unroll
        for (int j = 0; j < V; ++j) raw[j] = to_bits(o[j]);
        st_hint4(out + i0, raw, stream);
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
          if (i0 + j < n) out[i0 + j] = o[j];
      }
    }
    bar_workers<WT>();  // sm is reused; every worker has read its carry
    if (threadIdx.x == 0) st_release_shared(&cq_tail, it + 1);
  }
}

// ---- three kernels: block sums -> scan of block sums -> rescan --------------------------------
template <typename T, int OP, int THREADS, int V, int U>
__global__ void __launch_bounds__(THREADS)
scan_block_sums_kernel(const T* in, size_t n, size_t tiles_per_block, T* sums) {
  constexpr size_t TILE = size_t(THREADS) * V * U;
  __shared__ T smem[32];
  const T ident = identity<T, OP>();
  T acc = ident;
  const size_t t0 = size_t(blockIdx.x) * tiles_per_block;
  for (size_t t = t0; t < t0 + tiles_per_block; ++t) {
    const size_t base = t * TILE;
    if (base >= n) break;
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const size_t i0 = base + (size_t(u) * THREADS + threadIdx.x) * V;
      if (i0 + V <= n) {
        uint32_t raw[V];
        ld_stream<V, true>(raw, in + i0);
#pragma unroll
        for (int j = 0; j < V; ++j) acc = op2<T, OP>(acc, from_bits<T>(raw[j]));
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
          if (i0 + j < n) acc = op2<T, OP>(acc, in[i0 + j]);
      }
    }
  }
  acc = block_reduce<T, OP>(acc, smem);
  if (threadIdx.x == 0) sums[blockIdx.x] = acc;
}

// exclusive scan (seeded with `first`) of `count` block sums, in place, one block, fixed order
template <typename T, int OP>
__global__ void __launch_bounds__(256) scan_sums_kernel(T* sums, unsigned count, T first) {
  __shared__ T warp_tot[8];
  __shared__ T s_run;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const T ident = identity<T, OP>();
  if (threadIdx.x == 0) s_run = first;
  __syncthreads();
  for (unsigned base = 0; base < count; base += 256) {
    const unsigned i = base + threadIdx.x;
    const T v = i < count ? sums[i] : ident;
    T ws = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T y = __shfl_up_sync(FULL, ws, o);
      if (lane >= o) ws = op2<T, OP>(y, ws);
    }
    if (lane == 31) warp_tot[warp] = ws;
    __syncthreads();
    T wp = ident;
    for (int k = 0; k < warp; ++k) wp = op2<T, OP>(wp, warp_tot[k]);
    T ex = __shfl_up_sync(FULL, ws, 1);
    ex = lane == 0 ? ident : ex;
    const T run = s_run;
    if (i < count) sums[i] = op2<T, OP>(run, op2<T, OP>(wp, ex));
    __syncthreads();
    if (threadIdx.x == 255) s_run = op2<T, OP>(run, op2<T, OP>(wp, ws));
    __syncthreads();
  }
}

template <typename T, int OP, int THREADS, int V, int U, bool NC>
__global__ void __launch_bounds__(THREADS)
scan_rescan_kernel(const T* in, T* out, size_t n, size_t tiles_per_block, const T* carries, int exclusive) {
  constexpr int NW = THREADS / 32, E = U * NW;
  constexpr size_t TILE = size_t(THREADS) * V * U;
  __shared__ T sm[2 * E + 1];
  T carry = carries[blockIdx.x];
  const size_t t0 = size_t(blockIdx.x) * tiles_per_block;
  for (size_t t = t0; t < t0 + tiles_per_block; ++t) {
    const size_t base = t * TILE;
    if (base >= n) break;
    TileRegs<T, V, U> R;
    const T agg = tile_phase_a<T, OP, THREADS, V, U, NC>(in, base, n, R, sm);
    tile_phase_b<T, OP, THREADS, V, U>(out, base, n, R, sm, carry, exclusive != 0);
    carry = op2<T, OP>(carry, agg);
    __syncthreads();  // sm is reused by the next tile
  }
}

struct ScanVariant { const char* name; bool lookback; int threads, v, u; };
const ScanVariant kScanVariants[] = {
    {"lookback_256x4x4", true, 256, 4, 4},
    {"lookback_256x8x2", true, 256, 8, 2},
    {"lookback_512x8x2", true, 512, 8, 2},
    {"lookback_256x8x4", true, 256, 8, 4},
    {"three_kernel_256x4x4", false, 256, 4, 4},
    {"three_kernel_256x1x4", false, 256, 1, 4},  // any alignment
    {"lookback_512x8x4", true, 512, 8, 4},       // 16384-element tiles
    {"lookback_1024x8x2", true, 1024, 8, 2},     // 16384-element tiles, 1024 threads
    {"persist_256x8x4", true, 256, 8, 4},        // persistent blocks, strided tiles, no ticket
    {"persist_256x4x4", true, 256, 4, 4},
    {"persist_512x8x4", true, 512, 8, 4},
    {"ws_8w_u8_s6_k1", true, 256, 4, 8},         // warp-specialised: 32 KB tiles, 6 smem stages, 1 CTA/SM
    {"ws_8w_u8_s3_k2", true, 256, 4, 8},         // 32 KB tiles, 3 stages, 2 CTAs/SM
    {"ws_8w_u12_s4_k2", true, 256, 4, 12},       // 48 KB tiles, 4 stages
    {"l2ahead_8w_u4_d2_s2_b3", true, 256, 4, 4}, // TMA ring (S) -> reduce D tiles ahead -> scan re-reads from L2; 3 CTAs/SM
    {"l2ahead_8w_u8_d2_s2_b2", true, 256, 4, 8}, // 32 KB tiles, 2 CTAs/SM
    {"l2ahead_8w_u4_d3_s2_b3", true, 256, 4, 4},
    {"l2ahead_8w_u4_d2_s3_b3", true, 256, 4, 4},
};
constexpr int kNumScanVariants = sizeof(kScanVariants) / sizeof(kScanVariants[0]);

inline bool aligned_to(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

template <typename T, int OP, int THREADS, int V, int U>
cudaError_t launch_lookback(const Launch& L, Scratch& S, bool exclusive, T init, const T* in, T* out, size_t n) {
  constexpr size_t TILE = size_t(THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  if (ntiles > S.scan_state_tiles || ntiles > 0x7fffffffu) return cudaErrorInvalidValue;
  if (++S.scan_epoch >= (1u << 30)) {  // epoch wrap: start over from zeroed states
    cudaError_t e = cudaMemsetAsync(S.scan_state, 0, S.scan_state_tiles * 8, L.stream);
    if (e != cudaSuccess) return e;
    S.scan_epoch = 1;
  }
  const bool nc = static_cast<const void*>(in) != out;
  if (nc)
    scan_lookback_kernel<T, OP, THREADS, V, U, true><<<(unsigned)ntiles, THREADS, 0, L.stream>>>(
        in, out, n, init, exclusive ? 1 : 0, S.scan_state, S.scan_ticket, S.scan_epoch, (unsigned)ntiles);
  else
    scan_lookback_kernel<T, OP, THREADS, V, U, false><<<(unsigned)ntiles, THREADS, 0, L.stream>>>(
        in, out, n, init, exclusive ? 1 : 0, S.scan_state, S.scan_ticket, S.scan_epoch, (unsigned)ntiles);
  ++*L.launches;
  return cudaGetLastError();
}

template <typename T, int OP, int THREADS, int V, int U>
cudaError_t launch_persist(const Launch& L, Scratch& S, bool exclusive, T init, const T* in, T* out, size_t n) {
  constexpr size_t TILE = size_t(THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  if (ntiles > S.scan_state_tiles || ntiles > 0x7fffffffu) return cudaErrorInvalidValue;
  if (++S.scan_epoch >= (1u << 30)) {
    cudaError_t e = cudaMemsetAsync(S.scan_state, 0, S.scan_state_tiles * 8, L.stream);
    if (e != cudaSuccess) return e;
    S.scan_epoch = 1;
  }
  auto kt = scan_lookback_persist_kernel<T, OP, THREADS, V, U, true>;
  auto kf = scan_lookback_persist_kernel<T, OP, THREADS, V, U, false>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kf, THREADS, 0);
    if (e != cudaSuccess || per_sm < 1) return cudaErrorInvalidValue;
  }
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  const bool nc = static_cast<const void*>(in) != out;
  int excl = exclusive ? 1 : 0;
  uint32_t epoch = S.scan_epoch;
  unsigned nt = (unsigned)ntiles;
  void* args[] = {&in, &out, &n, &init, &excl, &S.scan_state, &epoch, &nt};
  // cooperative launch: the blocks wait on one another, so the driver must guarantee co-residency
  cudaError_t e = cudaLaunchCooperativeKernel(nc ? reinterpret_cast<void*>(kt) : reinterpret_cast<void*>(kf), dim3((unsigned)grid),
                                              dim3(THREADS), args, 0, L.stream);
  ++*L.launches;
  return e;
}

template <typename T, int OP, int NSW, int U, int S, int K>
cudaError_t launch_ws(const Launch& L, Scratch& Sc, bool exclusive, T init, const T* in, T* out, size_t n) {
  constexpr size_t TILE = size_t(NSW) * 32 * 4 * U;
  constexpr int THREADS = (NSW + S) * 32;
  constexpr size_t smem = S * TILE * 4 + 3 * S * 8 + S * NSW * 4 + 16;
  const size_t ntiles = (n + TILE - 1) / TILE;
  if (ntiles > Sc.scan_state_tiles || ntiles > 0x7fffffffu) return cudaErrorInvalidValue;
  if (++Sc.scan_epoch >= (1u << 30)) {
    cudaError_t e = cudaMemsetAsync(Sc.scan_state, 0, Sc.scan_state_tiles * 8, L.stream);
    if (e != cudaSuccess) return e;
    Sc.scan_epoch = 1;
  }
  auto kern = scan_ws_kernel<T, OP, NSW, U, S, K>;
  static int ctas_per_sm = 0;
  if (ctas_per_sm == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per < 1) return cudaErrorInvalidValue;
    ctas_per_sm = per;
  }
  size_t grid = size_t(L.sms) * ctas_per_sm;
  if (grid > ntiles) grid = ntiles;
  int excl = exclusive ? 1 : 0;
  uint32_t epoch = Sc.scan_epoch;
  unsigned nt = (unsigned)ntiles;
  void* args[] = {&in, &out, &n, &init, &excl, &Sc.scan_state, &epoch, &nt};
  cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void*>(kern), dim3((unsigned)grid), dim3(THREADS), args, smem, L.stream);
  ++*L.launches;
  return e;
}

template <typename T, int OP, int NW, int U, int D, int KW, int S, int MINB>
cudaError_t launch_l2(const Launch& L, Scratch& Sc, bool exclusive, T init, const T* in, T* out, size_t n) {
  constexpr size_t TILE = size_t(NW) * 32 * 4 * U;
  constexpr int THREADS = (NW + 1) * 32;
  constexpr size_t smem = S * TILE * 4 + S * 8 + 16;
  const size_t ntiles = (n + TILE - 1) / TILE;
  if (ntiles > Sc.scan_state_tiles || ntiles > 0x7fffffffu) return cudaErrorInvalidValue;
  if (++Sc.scan_epoch >= (1u << 30)) {
    cudaError_t e = cudaMemsetAsync(Sc.scan_state, 0, Sc.scan_state_tiles * 8, L.stream);
    if (e != cudaSuccess) return e;
    Sc.scan_epoch = 1;
  }
  auto kern = scan_l2_kernel<T, OP, NW, U, D, KW, S, MINB>;
  static int ctas_per_sm = 0;
  if (ctas_per_sm == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per < 1) return cudaErrorInvalidValue;
    ctas_per_sm = per;
  }
  size_t grid = size_t(L.sms) * ctas_per_sm;
  if (grid > ntiles) grid = ntiles;
  int excl = exclusive ? 1 : 0;
  uint32_t epoch = Sc.scan_epoch;
  unsigned nt = (unsigned)ntiles;
  void* args[] = {&in, &out, &n, &init, &excl, &Sc.scan_state, &epoch, &nt};
  cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void*>(kern), dim3((unsigned)grid), dim3(THREADS), args, smem, L.stream);
  ++*L.launches;
  return e;
}

template <typename T, int OP, int THREADS, int V, int U>
cudaError_t launch_three(const Launch& L, Scratch& S, bool exclusive, T init, const T* in, T* out, size_t n) {
  constexpr size_t TILE = size_t(THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  size_t grid = size_t(L.sms) * 8;
  if (grid > ntiles) grid = ntiles;
  if (grid > MAX_PARTIALS) grid = MAX_PARTIALS;
  const size_t tpb = (ntiles + grid - 1) / grid;
  grid = (ntiles + tpb - 1) / tpb;
  T* sums = static_cast<T*>(S.partials);
  T first;
  if (exclusive) first = init;
  else {
    // identity on the host side
    if (OP == FN_ADD) first = T(0);
    else if (OP == FN_MULT) first = T(1);
    else first = std::is_floating_point<T>::value ? T(-INFINITY) : T(INT32_MIN);
  }
  scan_block_sums_kernel<T, OP, THREADS, V, U><<<(unsigned)grid, THREADS, 0, L.stream>>>(in, n, tpb, sums);
  scan_sums_kernel<T, OP><<<1, 256, 0, L.stream>>>(sums, (unsigned)grid, first);
  const bool nc = static_cast<const void*>(in) != out;
  if (nc)
    scan_rescan_kernel<T, OP, THREADS, V, U, true><<<(unsigned)grid, THREADS, 0, L.stream>>>(in, out, n, tpb, sums, exclusive ? 1 : 0);
  else
    scan_rescan_kernel<T, OP, THREADS, V, U, false><<<(unsigned)grid, THREADS, 0, L.stream>>>(in, out, n, tpb, sums, exclusive ? 1 : 0);
  *L.launches += 3;
  return cudaGetLastError();
}

template <typename T, int OP>
cudaError_t launch_variant(const Launch& L, Scratch& S, int v, bool exclusive, T init, const T* in, T* out, size_t n) {
  if constexpr (std::is_same<T, int32_t>::value) {
    switch (v) {
      case 0: return launch_lookback<T, OP, 256, 4, 4>(L, S, exclusive, init, in, out, n);
      case 1: return launch_lookback<T, OP, 256, 8, 2>(L, S, exclusive, init, in, out, n);
      case 2: return launch_lookback<T, OP, 512, 8, 2>(L, S, exclusive, init, in, out, n);
      case 3: return launch_lookback<T, OP, 256, 8, 4>(L, S, exclusive, init, in, out, n);
      case 6: return launch_lookback<T, OP, 512, 8, 4>(L, S, exclusive, init, in, out, n);
      case 7: return launch_lookback<T, OP, 1024, 8, 2>(L, S, exclusive, init, in, out, n);
      case 8: return launch_persist<T, OP, 256, 8, 4>(L, S, exclusive, init, in, out, n);
      case 9: return launch_persist<T, OP, 256, 4, 4>(L, S, exclusive, init, in, out, n);
      case 10: return launch_persist<T, OP, 512, 8, 4>(L, S, exclusive, init, in, out, n);
      case 11: return launch_ws<T, OP, 8, 8, 6, 1>(L, S, exclusive, init, in, out, n);
      case 12: return launch_ws<T, OP, 8, 8, 3, 2>(L, S, exclusive, init, in, out, n);
      case 13: return launch_ws<T, OP, 8, 12, 4, 2>(L, S, exclusive, init, in, out, n);
      case 14: return launch_l2<T, OP, 8, 4, 2, 8, 2, 3>(L, S, exclusive, init, in, out, n);
      case 15: return launch_l2<T, OP, 8, 8, 2, 8, 2, 2>(L, S, exclusive, init, in, out, n);
      case 16: return launch_l2<T, OP, 8, 4, 3, 8, 2, 3>(L, S, exclusive, init, in, out, n);
      case 17: return launch_l2<T, OP, 8, 4, 2, 8, 3, 3>(L, S, exclusive, init, in, out, n);
    }
  }
  switch (v) {
    case 4: return launch_three<T, OP, 256, 4, 4>(L, S, exclusive, init, in, out, n);
    case 5: return launch_three<T, OP, 256, 1, 4>(L, S, exclusive, init, in, out, n);
  }
  return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t launch_op(const Launch& L, Scratch& S, int v, int op, bool exclusive, T init, const T* in, T* out, size_t n) {
  switch (op) {
    case FN_ADD: return launch_variant<T, FN_ADD>(L, S, v, exclusive, init, in, out, n);
    case FN_MULT: return launch_variant<T, FN_MULT>(L, S, v, exclusive, init, in, out, n);
    case FN_MAX: return launch_variant<T, FN_MAX>(L, S, v, exclusive, init, in, out, n);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

int scan_variant_count() { return kNumScanVariants; }
const char* scan_variant_name(int v) { return (v >= 0 && v < kNumScanVariants) ? kScanVariants[v].name : nullptr; }

bool scan_variant_ok(int v, int dtype, const void* in, const void* out, size_t) {
  if (v < 0 || v >= kNumScanVariants) return false;
  const ScanVariant& sv = kScanVariants[v];
  if (sv.lookback && dtype != DT_I32) return false;
  const size_t a = size_t(sv.v) * 4;
  return aligned_to(in, a) && aligned_to(out, a);  // (16 bytes for the ring variants' bulk copies: V == 4)
}

// smallest tile of any look-back variant is 4096 elements
size_t scan_tiles_needed(size_t n) { return (n + 4095) / 4096 + 1; }

cudaError_t launch_scan(const Launch& L, Scratch& S, int v, int dtype, int op, bool exclusive, uint32_t init_bits,
                        const void* in, void* out, size_t n) {
  if (n == 0) return cudaSuccess;
  if (dtype == DT_F32) {
    float init = __builtin_bit_cast(float, init_bits);
    return launch_op<float>(L, S, v, op, exclusive, init, static_cast<const float*>(in), static_cast<float*>(out), n);
  }
  return launch_op<int32_t>(L, S, v, op, exclusive, static_cast<int32_t>(init_bits), static_cast<const int32_t*>(in),
                            static_cast<int32_t*>(out), n);
}

}  // namespace skel
