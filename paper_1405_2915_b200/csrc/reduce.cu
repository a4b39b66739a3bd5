// Reduce and fused MapReduce skeletons (readings 2 and 3):
//   result = (+)_i f(in0[i], b_i)      f = identity for plain Reduce; the mapped value is never stored.
// One kernel: every thread folds its elements into V independent accumulators (128/256-bit
// streaming loads, U vectors per operand in flight), warp-shuffle + shared-memory block tree,
// one partial per block; the block that draws the last ticket folds the partials in a fixed order
// (bitwise deterministic for a given n and variant; no floating-point atomics). The ticket is an
// atomicInc that wraps to 0, so no memset is needed between calls. The "two_pass" variants write
// the partials and fold them in a second tiny kernel instead. The "chunk*" variants launch one block per contiguous
// chunk of the input (32 / 64 / 128 KB per operand, at most MAX_PARTIALS chunks) instead of 148 x k persistent blocks
// with a strided tile walk: the hardware block scheduler then balances the SMs (co-resident persistent blocks drift
// apart and an SM ends the kernel half empty), and the partial of a chunk depends on (n, variant) only: deterministic.
// The "*_iatom" variants replace the ticket + fold of an int32 ADD by ONE packed 64-bit atomicAdd per block (integer add
// is associative and commutative: the result has the same bits in any order): the running sum sits in the high 32 bits
// (wraps modulo 2^32), the count of arrived blocks in the low 32 bits, so a block pays a single L2 round trip, no fence
// and no partial; the block that reads count = grid - 1 holds the total and zeroes the word. Measured on B200 at
// n = 2^26: 43.3 us against 47.5 us for the fold in bench.py (46.0 -> 42-43 us back to back). The same idea for max
// (atomicMax on a scratch word + fence + ticket) was measured and dropped: two atomics per block on one 32-byte sector
// are 16 384 same-address atomics per launch, and their rate depends on where the scratch word lands (45.4 us in one
// process, 55.6 us in bench.py, against 47.5 us for the fold). Every other case (max, mult, fp32) takes the ordinary
// fold inside these variants.
// The "*_tag" variants keep the iatom end for an int32 ADD and end every other case WITHOUT a fence and without a
// wait: a block stores (partial bits, launch number) as ONE 64-bit relaxed.gpu word into its slot of a dedicated array
// (never cleared: the launch number never repeats within 2^32 launches) and exits. The ticket is drawn at the START of
// a block instead (its latency hides under the loads): the 8 blocks that STARTED last fold, each polling its eighth of
// the slots for this launch's number, and the very last one folds their 8 sub-totals (fold_tagged); every block they
// wait for is running or done or will start (8 waiting blocks never fill an SM), so the wait cannot deadlock. The fold
// order depends on (n, variant) only, like the ticket fold: bitwise deterministic. Measured on B200 at n = 2^26, back to
// back in one process: int32 max 46.3 -> 44.1 us, fp32 dot 88.5 -> 86.4 us (common.cuh holds fold_tagged: fused.cu
// ends its chain kernels the same way).
// `reverse` (chunk variants): block b takes chunk G - 1 - b, so the operand is walked from its end to its front; the
// partial's slot is the chunk's, so the result has the same bits (api.cu: L2-aware direction, skel_ctx_set_l2_reuse).
#include "common.cuh"
#include "kernels.hpp"
#include <string.h>
#include <type_traits>

namespace skel {
namespace {

constexpr int RED_THREADS = 256;

template <typename T, int OP>
__device__ __forceinline__ void fold_partials(const T* partials, unsigned count, T* result, T* smem) {
  T acc = identity<T, OP>();
  for (unsigned i = threadIdx.x; i < count; i += blockDim.x) acc = apply_fn<OP>(T(0), acc, partials[i]);
  __syncthreads();  // smem reuse
  acc = block_reduce<T, OP>(acc, smem);
  if (threadIdx.x == 0) *result = acc;
}

enum : int { END_PARTIALS = 0, END_FOLD = 1, END_ATOMIC = 2, END_TAGGED = 3 };

static_assert(TAG_SLOTS == MAX_PARTIALS, "the tagged slots mirror the partials");

// 8 blocks per SM = at most 32 registers, what the streaming loop of the 128-bit forms needs (2048 resident threads:
// the bytes in flight are what a 268 MB Reduce lives on; at 40 registers the int32 max fold lost 25 % of its warps and
// 0.8 us). Asked for where it costs no spill in the loop: one-operand V = 4 kernels and the tagged end.
template <typename T, int MAPF, bool HAS_IN1, int OP, int V, int U, int END>
__global__ void __launch_bounds__(RED_THREADS, ((V == 4 && !HAS_IN1) || END == END_TAGGED) ? 8 : 1)
mapreduce_kernel(const T* in0, const T* in1, T c, size_t n, T* partials, unsigned* ticket, T* result,
                 unsigned tiles_per_block /* 0: strided walk of a persistent grid; k: block b owns tiles b k .. b k + k - 1 */,
                 unsigned reverse /* chunk variants: the blocks take the chunks from the last one down (see launch_mapreduce) */,
                 unsigned long long* tagged = nullptr, uint32_t epoch = 0) {
  __shared__ T smem[32];
  __shared__ bool is_last;
  __shared__ unsigned s_order;
  unsigned order = 0;  // END_TAGGED, thread 0: this block's place in the order in which the blocks STARTED
  if constexpr (END == END_TAGGED) {
    if (threadIdx.x == 0 && gridDim.x > 1) order = atomicInc(ticket + 4, gridDim.x - 1);  // wraps to 0: self-resetting
  }
  constexpr size_t TILE = size_t(RED_THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  T acc[V];
#pragma unroll
  for (int j = 0; j < V; ++j) acc[j] = identity<T, OP>();

  // the chunk this block owns (= its partial's slot: the fold order does not depend on the direction)
  const unsigned chunk = (reverse && tiles_per_block) ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
  const size_t first = tiles_per_block ? size_t(chunk) * tiles_per_block : blockIdx.x;
  const size_t step = tiles_per_block ? 1 : gridDim.x;
  const size_t last = tiles_per_block ? (first + tiles_per_block < ntiles ? first + tiles_per_block : ntiles) : ntiles;
  for (size_t tile = first; tile < last; tile += step) {
    const size_t base = tile * TILE + size_t(threadIdx.x) * V;
    if (base + (U - 1) * size_t(RED_THREADS) * V + V <= n) {
      uint32_t a[U][V], b[U][V];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        ld_stream<V, true>(a[u], in0 + base + size_t(u) * RED_THREADS * V);
        if constexpr (HAS_IN1) ld_stream<V, true>(b[u], in1 + base + size_t(u) * RED_THREADS * V);
      }
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int j = 0; j < V; ++j) {
          T bv = HAS_IN1 ? from_bits<T>(b[u][j]) : c;
          acc[j] = apply_fn<OP>(T(0), acc[j], apply_fn<MAPF>(c, from_bits<T>(a[u][j]), bv));
        }
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const size_t i = base + size_t(u) * RED_THREADS * V + j;
          if (i < n) {
            T bv = HAS_IN1 ? in1[i] : c;
            acc[j] = apply_fn<OP>(T(0), acc[j], apply_fn<MAPF>(c, in0[i], bv));
          }
        }
    }
  }
  T v = acc[0];
#pragma unroll
  for (int j = 1; j < V; ++j) v = apply_fn<OP>(T(0), v, acc[j]);
  v = block_reduce<T, OP>(v, smem);

  if constexpr (END == END_ATOMIC) {  // int32 add only (launch_one)
    if (threadIdx.x == 0) {
      if (gridDim.x == 1) {
        *result = v;
      } else {
        unsigned long long* word = reinterpret_cast<unsigned long long*>(ticket + 2);
        const unsigned long long old = atomicAdd(word, ((unsigned long long)(uint32_t)v << 32) | 1ull);
        if (uint32_t(old) == gridDim.x - 1) {  // every other block has arrived: old carries their sum
          *result = T(uint32_t(old >> 32) + uint32_t(v));
          *word = 0;  // nobody else touches it in this launch; the next launch is ordered behind this one
        }
      }
    }
  } else if constexpr (END == END_TAGGED) {
    if (gridDim.x == 1) {
      if (threadIdx.x == 0) *result = v;
      return;
    }
    if (threadIdx.x == 0) {
      // partial and launch number in ONE 64-bit store: no fence, nothing to wait for
      const unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned long long)to_bits(v);
      asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(tagged + chunk), "l"(w) : "memory");
      s_order = order;
    }
    __syncthreads();
    const unsigned ord = s_order;
    if (ord + TAG_P >= gridDim.x) fold_tagged<T, OP, RED_THREADS>(tagged, gridDim.x, ord, epoch, result, smem);
  } else if constexpr (END == END_FOLD) {
    if (gridDim.x == 1) {
      if (threadIdx.x == 0) *result = v;
      return;
    }
    if (threadIdx.x == 0) {
      partials[chunk] = v;
      __threadfence();
      const unsigned t = atomicInc(ticket, gridDim.x - 1);  // wraps back to 0 on the last arrival
      is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
      __threadfence();
      fold_partials<T, OP>(partials, gridDim.x, result, smem);
    }
  } else {
    if (threadIdx.x == 0) partials[chunk] = v;
  }
}

template <typename T, int OP>
__global__ void __launch_bounds__(RED_THREADS) fold_kernel(const T* partials, unsigned count, T* result) {
  __shared__ T smem[32];
  fold_partials<T, OP>(partials, count, result, smem);
}

struct RedVariant { const char* name; int v, u; bool single; int blocks_per_sm; unsigned chunk_bytes = 0; bool iatom = false; bool tagged = false; };
const RedVariant kRedVariants[] = {
    {"scalar_single_pass", 1, 4, true, 8},
    {"v4_u4_single_pass", 4, 4, true, 8},
    {"v8_u2_single_pass", 8, 2, true, 8},
    {"v4_u4_two_pass", 4, 4, false, 8},
    {"v8_u2_two_pass", 8, 2, false, 8},
    {"v4_u4_single_pass_4bps", 4, 4, true, 4},
    {"v4_u4_chunk32k", 4, 4, true, 0, 32768},
    {"v4_u4_chunk64k", 4, 4, true, 0, 65536},
    {"v4_u4_chunk128k", 4, 4, true, 0, 131072},
    {"v8_u2_chunk64k", 8, 2, true, 0, 65536},
    {"v4_u4_chunk32k_iatom", 4, 4, true, 0, 32768, true},
    {"v4_u4_chunk64k_iatom", 4, 4, true, 0, 65536, true},
    {"v4_u4_chunk32k_tag", 4, 4, true, 0, 32768, true, true},
    {"v4_u4_chunk64k_tag", 4, 4, true, 0, 65536, true, true},
};
constexpr int kNumRedVariants = sizeof(kRedVariants) / sizeof(kRedVariants[0]);

inline bool aligned_to(const void* p, size_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) % a) == 0; }

template <typename T, int MAPF, bool HAS_IN1, int OP, int V, int U>
cudaError_t launch_one(const Launch& L, const Scratch& S, const RedVariant& rv, const T* in0, const T* in1, T c,
                       size_t n, T* result, unsigned rev) {
  constexpr size_t TILE = size_t(RED_THREADS) * V * U;
  size_t ntiles = (n + TILE - 1) / TILE;
  size_t grid = size_t(L.sms) * rv.blocks_per_sm;
  unsigned tpb = 0;
  if (rv.chunk_bytes) {  // one block per chunk; chunks grow when there would be more than MAX_PARTIALS of them
    size_t t = rv.chunk_bytes / (TILE * sizeof(T));
    if (t < 1) t = 1;
    const size_t need = (ntiles + MAX_PARTIALS - 1) / MAX_PARTIALS;
    if (t < need) t = need;
    tpb = (unsigned)t;
    grid = (ntiles + t - 1) / t;
  }
  if (grid > ntiles) grid = ntiles;
  if (grid > MAX_PARTIALS) grid = MAX_PARTIALS;
  T* partials = static_cast<T*>(S.partials);
  if constexpr (std::is_same<T, int32_t>::value && OP == FN_ADD && V == 4) {
    if (rv.iatom) {
      mapreduce_kernel<T, MAPF, HAS_IN1, OP, V, U, END_ATOMIC>
          <<<(unsigned)grid, RED_THREADS, 0, L.stream>>>(in0, in1, c, n, partials, S.ticket, result, tpb, rev);
      ++*L.launches;
      return cudaGetLastError();
    }
  }
  if constexpr (V == 4) {
    if (rv.tagged) {
      if (++S.red_epoch == 0) {  // 2^32 launches: start over from cleared slots
        cudaError_t e = cudaMemsetAsync(S.red_tagged, 0, size_t(MAX_PARTIALS + 8) * 8, L.stream);
        if (e != cudaSuccess) return e;
        S.red_epoch = 1;
      }
      mapreduce_kernel<T, MAPF, HAS_IN1, OP, V, U, END_TAGGED>
          <<<(unsigned)grid, RED_THREADS, 0, L.stream>>>(in0, in1, c, n, partials, S.ticket, result, tpb, rev, S.red_tagged, S.red_epoch);
      ++*L.launches;
      return cudaGetLastError();
    }
  }
  if (rv.single) {
    mapreduce_kernel<T, MAPF, HAS_IN1, OP, V, U, END_FOLD>
        <<<(unsigned)grid, RED_THREADS, 0, L.stream>>>(in0, in1, c, n, partials, S.ticket, result, tpb, rev);
    ++*L.launches;
  } else {
    mapreduce_kernel<T, MAPF, HAS_IN1, OP, V, U, END_PARTIALS>
        <<<(unsigned)grid, RED_THREADS, 0, L.stream>>>(in0, in1, c, n, partials, S.ticket, result, tpb, rev);
    fold_kernel<T, OP><<<1, RED_THREADS, 0, L.stream>>>(partials, (unsigned)grid, result);
    *L.launches += 2;
  }
  return cudaGetLastError();
}

template <typename T, int MAPF, bool HAS_IN1, int OP>
cudaError_t launch_vu(const Launch& L, const Scratch& S, const RedVariant& rv, const T* in0, const T* in1, T c,
                      size_t n, T* result, unsigned rev) {
  if (rv.v == 1) return launch_one<T, MAPF, HAS_IN1, OP, 1, 4>(L, S, rv, in0, in1, c, n, result, rev);
  if (rv.v == 4) return launch_one<T, MAPF, HAS_IN1, OP, 4, 4>(L, S, rv, in0, in1, c, n, result, rev);
  return launch_one<T, MAPF, HAS_IN1, OP, 8, 2>(L, S, rv, in0, in1, c, n, result, rev);
}

template <typename T, int MAPF, bool HAS_IN1>
cudaError_t launch_op(const Launch& L, const Scratch& S, const RedVariant& rv, int op, const T* in0, const T* in1,
                      T c, size_t n, T* result, unsigned rev) {
  switch (op) {
    case FN_ADD: return launch_vu<T, MAPF, HAS_IN1, FN_ADD>(L, S, rv, in0, in1, c, n, result, rev);
    case FN_MULT: return launch_vu<T, MAPF, HAS_IN1, FN_MULT>(L, S, rv, in0, in1, c, n, result, rev);
    case FN_MAX: return launch_vu<T, MAPF, HAS_IN1, FN_MAX>(L, S, rv, in0, in1, c, n, result, rev);
  }
  return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t launch_t(const Launch& L, const Scratch& S, const RedVariant& rv, int map_fn, bool has_in1, int op,
                     T c, const T* in0, const T* in1, size_t n, T* result, unsigned rev) {
#define SKEL_MR_CASE(F)                                                                   \
  case F:                                                                                 \
    return has_in1 ? launch_op<T, F, true>(L, S, rv, op, in0, in1, c, n, result, rev)     \
                   : launch_op<T, F, false>(L, S, rv, op, in0, in1, c, n, result, rev);
  switch (map_fn) {
    case FN_IDENT: return launch_op<T, FN_IDENT, false>(L, S, rv, op, in0, in1, c, n, result, rev);
    SKEL_MR_CASE(FN_ADD)
    SKEL_MR_CASE(FN_MULT)
    SKEL_MR_CASE(FN_MAX)
    case FN_SAXPY: return launch_op<T, FN_SAXPY, true>(L, S, rv, op, in0, in1, c, n, result, rev);
  }
#undef SKEL_MR_CASE
  return cudaErrorInvalidValue;
}

// ---- row-wise Reduce on a matrix: out[i] = in[i][0] (+) ... (+) in[i][cols-1] --------
// "warp_*": one warp per row (8 rows per block): a lane folds its V-wide vectors into 4 x V independent chains
// (4 vectors in flight), then a fixed shuffle tree; "block_v4": 256 threads per row (long rows, few of them), 16 x 148
// persistent blocks; "block_v4_row": the same kernel with one block per row.
// The combination order depends only on (cols, variant): deterministic run to run.
template <typename T, int OP, int V>
__device__ __forceinline__ T fold_row_part(const T* row, size_t cols, int t, int nt) {
  // thread t of nt cooperating threads folds the vectors t, t + nt, t + 2 nt, ... of the row
  constexpr int U = 4;
  T acc[U][V];
#pragma unroll
  for (int u = 0; u < U; ++u)
#pragma unroll
    for (int j = 0; j < V; ++j) acc[u][j] = identity<T, OP>();
  const size_t nvec = cols / V;
  size_t i = t;
  for (; i + size_t(U - 1) * nt < nvec; i += size_t(U) * nt) {
    uint32_t raw[U][V];
#pragma unroll
    for (int u = 0; u < U; ++u) ld_stream<V, true>(raw[u], row + (i + size_t(u) * nt) * V);
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int j = 0; j < V; ++j) acc[u][j] = apply_fn<OP>(T(0), acc[u][j], from_bits<T>(raw[u][j]));
  }
  for (; i < nvec; i += nt) {
    uint32_t raw[V];
    ld_stream<V, true>(raw, row + i * V);
#pragma unroll
    for (int j = 0; j < V; ++j) acc[0][j] = apply_fn<OP>(T(0), acc[0][j], from_bits<T>(raw[j]));
  }
  for (size_t c = nvec * V + t; c < cols; c += nt) acc[1][0] = apply_fn<OP>(T(0), acc[1][0], row[c]);  // V > 1: ragged tail
  T v = identity<T, OP>();
#pragma unroll
  for (int u = 0; u < U; ++u)
#pragma unroll
    for (int j = 0; j < V; ++j) v = apply_fn<OP>(T(0), v, acc[u][j]);
  return v;
}

template <typename T, int OP, int V>
__global__ void __launch_bounds__(RED_THREADS)
reduce_rows_warp_kernel(const T* in, size_t rows, size_t cols, T* out) {
  const int lane = threadIdx.x & 31;
  const size_t warps_per_grid = size_t(gridDim.x) * (RED_THREADS / 32);
  for (size_t row = size_t(blockIdx.x) * (RED_THREADS / 32) + (threadIdx.x >> 5); row < rows; row += warps_per_grid) {
    T v = fold_row_part<T, OP, V>(in + row * cols, cols, lane, 32);
    v = warp_reduce<T, OP>(v);
    if (lane == 0) out[row] = v;
  }
}

template <typename T, int OP, int V>
__global__ void __launch_bounds__(RED_THREADS)
reduce_rows_block_kernel(const T* in, size_t rows, size_t cols, T* out) {
  __shared__ T smem[32];
  for (size_t row = blockIdx.x; row < rows; row += gridDim.x) {
    T v = fold_row_part<T, OP, V>(in + row * cols, cols, threadIdx.x, RED_THREADS);
    v = block_reduce<T, OP>(v, smem);
    if (threadIdx.x == 0) out[row] = v;
    __syncthreads();  // smem is reused by the next row
  }
}

const char* const kRowNames[] = {"warp_scalar", "warp_v4", "block_v4", "block_v4_row"};
constexpr int kNumRowVariants = 4;

template <typename T, int OP>
cudaError_t launch_rows_op(const Launch& L, int v, const T* in, size_t rows, size_t cols, T* out) {
  const size_t cap = size_t(L.sms) * 16;
  if (v == 3) {  // one block per row: the hardware block scheduler balances the SMs (like Reduce's chunk variants)
    const unsigned grid = (unsigned)(rows < 0x7fffffffu ? rows : 0x7fffffffu);
    reduce_rows_block_kernel<T, OP, 4><<<grid, RED_THREADS, 0, L.stream>>>(in, rows, cols, out);
  } else if (v == 2) {
    const unsigned grid = (unsigned)(rows < cap ? rows : cap);
    reduce_rows_block_kernel<T, OP, 4><<<grid, RED_THREADS, 0, L.stream>>>(in, rows, cols, out);
  } else {
    const size_t blocks = (rows + RED_THREADS / 32 - 1) / (RED_THREADS / 32);
    const unsigned grid = (unsigned)(blocks < cap ? blocks : cap);
    if (v == 1) reduce_rows_warp_kernel<T, OP, 4><<<grid, RED_THREADS, 0, L.stream>>>(in, rows, cols, out);
    else reduce_rows_warp_kernel<T, OP, 1><<<grid, RED_THREADS, 0, L.stream>>>(in, rows, cols, out);
  }
  ++*L.launches;
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_rows_t(const Launch& L, int v, int op, const T* in, size_t rows, size_t cols, T* out) {
  switch (op) {
    case FN_ADD: return launch_rows_op<T, FN_ADD>(L, v, in, rows, cols, out);
    case FN_MULT: return launch_rows_op<T, FN_MULT>(L, v, in, rows, cols, out);
    case FN_MAX: return launch_rows_op<T, FN_MAX>(L, v, in, rows, cols, out);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

int reduce_rows_variant_count() { return kNumRowVariants; }
const char* reduce_rows_variant_name(int v) { return (v >= 0 && v < kNumRowVariants) ? kRowNames[v] : nullptr; }
bool reduce_rows_variant_ok(int v, const void* in, size_t, size_t cols) {
  if (v < 0 || v >= kNumRowVariants) return false;
  if (v == 0) return true;
  return aligned_to(in, 16) && cols % 4 == 0;  // every row starts on a 16-byte boundary
}
cudaError_t launch_reduce_rows(const Launch& L, int v, int dtype, int op, const void* in, size_t rows, size_t cols,
                               void* out) {
  if (rows == 0) return cudaSuccess;
  if (dtype == DT_F32)
    return launch_rows_t<float>(L, v, op, static_cast<const float*>(in), rows, cols, static_cast<float*>(out));
  return launch_rows_t<int32_t>(L, v, op, static_cast<const int32_t*>(in), rows, cols, static_cast<int32_t*>(out));
}

int reduce_variant_count() { return kNumRedVariants; }
const char* reduce_variant_name(int v) { return (v >= 0 && v < kNumRedVariants) ? kRedVariants[v].name : nullptr; }

bool reduce_variant_ok(int v, const void* in0, const void* in1, size_t) {
  if (v < 0 || v >= kNumRedVariants) return false;
  const size_t a = size_t(kRedVariants[v].v) * 4;
  return aligned_to(in0, a) && aligned_to(in1, a);
}

cudaError_t launch_mapreduce(const Launch& L, const Scratch& S, int v, int dtype, int map_fn, bool has_in1,
                             int red_op, uint32_t cbits, const void* in0, const void* in1, size_t n, void* result,
                             bool reverse) {
  const RedVariant& rv = kRedVariants[v];
  const unsigned rev = reverse ? 1u : 0u;
  if (dtype == DT_F32) {
    float c;
    memcpy(&c, &cbits, 4);
    return launch_t<float>(L, S, rv, map_fn, has_in1, red_op, c, static_cast<const float*>(in0),
                           static_cast<const float*>(in1), n, static_cast<float*>(result), rev);
  }
  return launch_t<int32_t>(L, S, rv, map_fn, has_in1, red_op, static_cast<int32_t>(cbits),
                           static_cast<const int32_t*>(in0), static_cast<const int32_t*>(in1), n,
                           static_cast<int32_t*>(result), rev);
}

}  // namespace skel
