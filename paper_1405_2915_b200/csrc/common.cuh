// Device-side helpers shared by the skeleton kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace skel {

// user-function ids: same values as skel_fn in include/skel.h
enum : int { FN_ADD = 0, FN_MULT = 1, FN_MAX = 2, FN_SAXPY = 3, FN_IDENT = 100 };

// ---- streaming 32/128/256-bit global accesses ------------------------------------------------
// NC = true uses the non-coherent path (only legal when the kernel never writes the buffer, i.e.
// not for in-place calls). L1::no_allocate: every skeleton input is touched once per call.
template <int V, bool NC>
__device__ __forceinline__ void ld_stream(uint32_t (&r)[V], const void* p) {
  static_assert(V == 1 || V == 2 || V == 4 || V == 8, "vector width");
  if constexpr (V == 8) {
    if constexpr (NC)
      asm volatile("ld.global.nc.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                   : "l"(p));
    else
      asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                   : "l"(p)
                   : "memory");
  } else if constexpr (V == 4) {
    if constexpr (NC)
      asm volatile("ld.global.nc.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                   : "l"(p));
    else
      asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                   : "l"(p)
                   : "memory");
  } else if constexpr (V == 2) {
    if constexpr (NC)
      asm volatile("ld.global.nc.L1::no_allocate.v2.b32 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "l"(p));
    else
      asm volatile("ld.global.L1::no_allocate.v2.b32 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "l"(p) : "memory");
  } else {
    if constexpr (NC)
      asm volatile("ld.global.nc.L1::no_allocate.b32 %0, [%1];" : "=r"(r[0]) : "l"(p));
    else
      asm volatile("ld.global.L1::no_allocate.b32 %0, [%1];" : "=r"(r[0]) : "l"(p) : "memory");
  }
}

template <int V>
__device__ __forceinline__ void st_stream(void* p, const uint32_t (&r)[V]) {
  static_assert(V == 1 || V == 2 || V == 4 || V == 8, "vector width");
  if constexpr (V == 8)
    asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
  else if constexpr (V == 4)
    asm volatile("st.global.L1::no_allocate.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(r[0]), "r"(r[1]), "r"(r[2]),
                 "r"(r[3])
                 : "memory");
  else if constexpr (V == 2)
    asm volatile("st.global.L1::no_allocate.v2.b32 [%0], {%1,%2};" ::"l"(p), "r"(r[0]), "r"(r[1]) : "memory");
  else
    asm volatile("st.global.L1::no_allocate.b32 [%0], %1;" ::"l"(p), "r"(r[0]) : "memory");
}

// ---- 128-bit global accesses with an L2 eviction-priority policy ---------------------------------
// evict_last: "I will read this line again soon" (kept in L2); evict_first: touch-once streaming.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void ld_hint4(uint32_t (&r)[4], const void* p, uint64_t policy) {
  asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.b32 {%0,%1,%2,%3}, [%4], %5;"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "l"(p), "l"(policy)
               : "memory");
}
__device__ __forceinline__ void st_hint4(void* p, const uint32_t (&r)[4], uint64_t policy) {
  asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.b32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(r[0]), "r"(r[1]),
               "r"(r[2]), "r"(r[3]), "l"(policy)
               : "memory");
}

// ---- mbarrier + bulk async copy (TMA engine, 1-D form; SASS: UBLKCP / SYNCS) ---------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// global -> shared bulk copy; completion is signalled on `bar` (complete_tx of `bytes`).
// src, dst 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// the same with an L2 eviction-priority policy (createpolicy)
__device__ __forceinline__ void bulk_load_hint(void* smem_dst, const void* gsrc, unsigned bytes, uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(smem_dst)),
      "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// ---- bit casts between the 32-bit register image and the element type ---------------------------
template <typename T> __device__ __forceinline__ T from_bits(uint32_t b);
template <> __device__ __forceinline__ float from_bits<float>(uint32_t b) { return __uint_as_float(b); }
template <> __device__ __forceinline__ int32_t from_bits<int32_t>(uint32_t b) { return static_cast<int32_t>(b); }
__device__ __forceinline__ uint32_t to_bits(float v) { return __float_as_uint(v); }
__device__ __forceinline__ uint32_t to_bits(int32_t v) { return static_cast<uint32_t>(v); }

// ---- user functions --------------------------------------------------------------------------
// f32: add/mult are correctly rounded; saxpy is ONE fused multiply-add (reading 4);
// i32: two's-complement wrap-around (computed on uint32_t, reading 7).
template <int FN> __device__ __forceinline__ float apply_fn(float c, float a, float b) {
  if constexpr (FN == FN_ADD) return __fadd_rn(a, b);
  else if constexpr (FN == FN_MULT) return __fmul_rn(a, b);
  else if constexpr (FN == FN_MAX) return a < b ? b : a;
  else if constexpr (FN == FN_SAXPY) return __fmaf_rn(c, a, b);
  else return a;  // FN_IDENT
}
template <int FN> __device__ __forceinline__ int32_t apply_fn(int32_t c, int32_t a, int32_t b) {
  if constexpr (FN == FN_ADD) return static_cast<int32_t>(static_cast<uint32_t>(a) + static_cast<uint32_t>(b));
  else if constexpr (FN == FN_MULT) return static_cast<int32_t>(static_cast<uint32_t>(a) * static_cast<uint32_t>(b));
  else if constexpr (FN == FN_MAX) return a < b ? b : a;
  else if constexpr (FN == FN_SAXPY)
    return static_cast<int32_t>(static_cast<uint32_t>(c) * static_cast<uint32_t>(a) + static_cast<uint32_t>(b));
  else return a;
}

// ---- MapOverlap element arithmetic ---------------------------------------------------------------
// The stencil kernels move 32-bit register images typed `float` whatever the element type (loads, shared memory, TMA,
// shuffles and stores do not look at the bits); only the multiply-add of a tap and the addition of two partial sums
// interpret them. f32: one fused multiply-add (FFMA); i32: multiply-add modulo 2^32 on uint32_t (IMAD), DESIGN.md
// reading 26. The packed FFMA2 forms exist for f32 only.
template <typename T> struct StencilOps;
template <> struct StencilOps<float> {
  static constexpr bool kFloat = true;
  static __device__ __forceinline__ float mad(float w, float x, float acc) { return fmaf(w, x, acc); }
  static __device__ __forceinline__ float add(float a, float b) { return a + b; }
};
template <> struct StencilOps<int32_t> {
  static constexpr bool kFloat = false;
  static __device__ __forceinline__ float mad(float w, float x, float acc) {
    return __uint_as_float(__float_as_uint(w) * __float_as_uint(x) + __float_as_uint(acc));
  }
  static __device__ __forceinline__ float add(float a, float b) { return __uint_as_float(__float_as_uint(a) + __float_as_uint(b)); }
};
__device__ __forceinline__ bool bits_are_zero(float v) { return __float_as_uint(v) == 0u; }

// identity element of a reduction operator
template <typename T, int OP> __device__ __forceinline__ T identity() {
  if constexpr (OP == FN_ADD) return T(0);
  else if constexpr (OP == FN_MULT) return T(1);
  else {
    if constexpr (std::is_floating_point<T>::value) return T(-INFINITY);
    else return T(INT32_MIN);
  }
}

template <typename T, int OP> __device__ __forceinline__ T warp_reduce(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = apply_fn<OP>(T(0), v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Block-wide reduction; result valid in thread 0. `smem` holds >= 32 elements of T.
// The combination order is fixed by (blockDim, lane, warp): deterministic run to run.
template <typename T, int OP> __device__ __forceinline__ T block_reduce(T v, T* smem) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
  v = warp_reduce<T, OP>(v);
  if (lane == 0) smem[warp] = v;
  __syncthreads();
  if (warp == 0) {
    v = lane < nwarps ? smem[lane] : identity<T, OP>();
    v = warp_reduce<T, OP>(v);
  }
  return v;
}

// ---- the tagged end of the reducing kernels (reduce.cu END_TAGGED, fused.cu) ----------------------------------------
// 128-bit relaxed.gpu load of two (partial bits, launch number) slots
__device__ __forceinline__ void ld_tagged2(const unsigned long long* p, unsigned long long& w0, unsigned long long& w1) {
  asm volatile("{\n.reg .b128 t;\nld.relaxed.gpu.global.b128 t, [%2];\nmov.b128 {%0, %1}, t;\n}"
               : "=l"(w0), "=l"(w1) : "l"(p) : "memory");
}

// The end of END_TAGGED in two levels. The TAG_P blocks that STARTED last are the pollers: poller j waits for the slots
// j S .. j S + S - 1 (S = slots per poller, fixed by the grid) to carry this launch's number, folds them in index order
// (thread t takes the slot pairs t, t + NT, ...; then the block tree) and publishes the sub-total the same way in the
// second-level slot j; the block that started LAST also waits for the TAG_P second-level slots and folds them in index
// order. A thread has one 128-bit load in flight per step (a poller reads at most 1024 slots at the usual grids), so the
// kernel keeps the 32 registers of the streaming loop. Every block stores its own slot BEFORE it waits and at most TAG_P
// = 8 blocks wait, fewer than the device holds at once (reduce.cu: 8 per SM by __launch_bounds__(256, 8); fused.cu: 3 or
// more per SM on 148 SMs), so a block that has not started yet always finds a slot: the waits cannot deadlock. Grouping
// and order depend on (gridDim) only: the same bits on every run.
constexpr unsigned TAG_P = 8;
constexpr unsigned TAG_SLOTS = 8192;  // per-block slots (as many as Reduce partials, kernels.hpp); the TAG_P second-level slots follow them

template <typename T, int OP, int NT /* threads per block */>
__device__ __forceinline__ void fold_tagged(unsigned long long* tagged, unsigned count, unsigned order, uint32_t epoch,
                                            T* result, T* smem) {
  unsigned long long* level2 = tagged + TAG_SLOTS;  // TAG_P slots behind the per-block slots
  const unsigned P = count < TAG_P ? count : TAG_P;
  const unsigned j = order - (count - P);                      // this poller's index, 0 .. P - 1
  const unsigned per = (((count + P - 1) / P) + 1) & ~1u;      // slots per poller, even: a pair never straddles two pollers
  const unsigned lo = j * per;
  const unsigned hi = lo + per < count ? lo + per : count;
  T acc = identity<T, OP>();
  for (unsigned s0 = lo + 2 * threadIdx.x; s0 < hi; s0 += 2 * NT) {
    unsigned long long w0, w1;
    bool ok;
    do {
      ld_tagged2(tagged + s0, w0, w1);
      ok = uint32_t(w0 >> 32) == epoch && (s0 + 1 >= hi || uint32_t(w1 >> 32) == epoch);
    } while (!ok);
    acc = apply_fn<OP>(T(0), acc, from_bits<T>(uint32_t(w0)));
    if (s0 + 1 < hi) acc = apply_fn<OP>(T(0), acc, from_bits<T>(uint32_t(w1)));
  }
  __syncthreads();  // smem reuse
  acc = block_reduce<T, OP>(acc, smem);
  if (threadIdx.x == 0) {
    const unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned long long)to_bits(acc);
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(level2 + j), "l"(w) : "memory");
  }
  if (order != count - 1 || threadIdx.x >= 32) return;
  // the block that started last: second level, lanes 0 .. P - 1 of warp 0
  T v = identity<T, OP>();
  if (threadIdx.x < P) {
    unsigned long long w;
    do {
      asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(level2 + threadIdx.x) : "memory");
    } while (uint32_t(w >> 32) != epoch);
    v = from_bits<T>(uint32_t(w));
  }
  v = warp_reduce<T, OP>(v);
  if (threadIdx.x == 0) *result = v;
}

}  // namespace skel
