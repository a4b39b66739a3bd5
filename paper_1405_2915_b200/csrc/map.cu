// Map skeleton (PAPER.md L75/L83 name it; definition: DESIGN.md reading 1):
//   out[i] = f(in0[i], b_i),  b_i = in1[i] or the constant c.
// HBM-bound (8-12 B/elem): 128/256-bit streaming loads, all loads of a tile issued before the
// first use (U vectors per operand in flight per thread), L1 no-allocate, no shared memory.
#include "common.cuh"
#include "kernels.hpp"
#include <string.h>

namespace skel {
namespace {

constexpr int MAP_THREADS = 256;

// One tile = MAP_THREADS * V * U consecutive elements; inside a tile, vector u of thread t sits at
// (u * MAP_THREADS + t) * V so that a warp's accesses are contiguous. Grid-stride over tiles: the
// "tiles" variants launch one block per tile, the "persist" variants a multiple of the SM count.
template <typename T, int FN, bool HAS_IN1, int V, int U, bool NC>
__global__ void __launch_bounds__(MAP_THREADS)
map_kernel(const T* in0, const T* in1, T* out, T c, size_t n) {
  constexpr size_t TILE = size_t(MAP_THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t base = tile * TILE + size_t(threadIdx.x) * V;
    if (base + (U - 1) * size_t(MAP_THREADS) * V + V <= n) {  // all U vectors of this thread in range
      uint32_t a[U][V], b[U][V];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        ld_stream<V, NC>(a[u], in0 + base + size_t(u) * MAP_THREADS * V);
        if constexpr (HAS_IN1) ld_stream<V, NC>(b[u], in1 + base + size_t(u) * MAP_THREADS * V);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
#pragma unroll
        for (int j = 0; j < V; ++j) {
          T bv = HAS_IN1 ? from_bits<T>(b[u][j]) : c;
          a[u][j] = to_bits(apply_fn<FN>(c, from_bits<T>(a[u][j]), bv));
        }
        st_stream<V>(out + base + size_t(u) * MAP_THREADS * V, a[u]);
      }
    } else {  // ragged end of the last tile: element-wise
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const size_t i0 = base + size_t(u) * MAP_THREADS * V;
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const size_t i = i0 + j;
          if (i < n) {
            T bv = HAS_IN1 ? in1[i] : c;
            out[i] = apply_fn<FN>(c, in0[i], bv);
          }
        }
      }
    }
  }
}

// Three-vector Map, MULADD: out[i] = in0[i] * in1[i] + in2[i] (f32: ONE fused multiply-add, like
// saxpy; i32 wraps). 16 B/elem; same tile layout, U2 = 2 vectors per operand in flight (three operands).
template <typename T, int V, int U, bool NC>
__global__ void __launch_bounds__(MAP_THREADS)
map3_kernel(const T* in0, const T* in1, const T* in2, T* out, size_t n) {
  constexpr size_t TILE = size_t(MAP_THREADS) * V * U;
  const size_t ntiles = (n + TILE - 1) / TILE;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t base = tile * TILE + size_t(threadIdx.x) * V;
    if (base + (U - 1) * size_t(MAP_THREADS) * V + V <= n) {
      uint32_t a[U][V], b[U][V], c[U][V];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        ld_stream<V, NC>(a[u], in0 + base + size_t(u) * MAP_THREADS * V);
        ld_stream<V, NC>(b[u], in1 + base + size_t(u) * MAP_THREADS * V);
        ld_stream<V, NC>(c[u], in2 + base + size_t(u) * MAP_THREADS * V);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
#pragma unroll
        for (int j = 0; j < V; ++j)  // saxpy's arithmetic with a per-element factor: c' * a + b with c' = in0, a = in1, b = in2
          a[u][j] = to_bits(apply_fn<FN_SAXPY>(from_bits<T>(a[u][j]), from_bits<T>(b[u][j]), from_bits<T>(c[u][j])));
        st_stream<V>(out + base + size_t(u) * MAP_THREADS * V, a[u]);
      }
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const size_t i0 = base + size_t(u) * MAP_THREADS * V;
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const size_t i = i0 + j;
          if (i < n) out[i] = apply_fn<FN_SAXPY>(in0[i], in1[i], in2[i]);
        }
      }
    }
  }
}

struct MapVariant { const char* name; int v, u; bool persist; };
const MapVariant kMapVariants[] = {
    {"scalar_u4_tiles", 1, 4, false},   // any alignment
    {"v4_u4_tiles", 4, 4, false},       // 128-bit accesses
    {"v8_u2_tiles", 8, 2, false},       // 256-bit accesses
    {"v4_u4_persist", 4, 4, true},
    {"v8_u2_persist", 8, 2, true},
    {"v8_u4_tiles", 8, 4, false},
};
constexpr int kNumMapVariants = sizeof(kMapVariants) / sizeof(kMapVariants[0]);

inline bool aligned_to(const void* p, size_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) % a) == 0; }

template <typename T, int FN, bool HAS_IN1, int V, int U>
cudaError_t launch_one(const Launch& L, bool persist, bool nc, const T* in0, const T* in1, T* out, T c, size_t n) {
  constexpr size_t TILE = size_t(MAP_THREADS) * V * U;
  size_t ntiles = (n + TILE - 1) / TILE;
  size_t grid = persist ? (size_t)L.sms * 8 : ntiles;
  if (grid > ntiles) grid = ntiles;
  if (grid > 0x7fffffffu) grid = 0x7fffffffu;
  if (nc) map_kernel<T, FN, HAS_IN1, V, U, true><<<(unsigned)grid, MAP_THREADS, 0, L.stream>>>(in0, in1, out, c, n);
  else map_kernel<T, FN, HAS_IN1, V, U, false><<<(unsigned)grid, MAP_THREADS, 0, L.stream>>>(in0, in1, out, c, n);
  ++*L.launches;
  return cudaGetLastError();
}

template <typename T, int FN, bool HAS_IN1>
cudaError_t launch_vu(const Launch& L, const MapVariant& mv, bool nc, const T* in0, const T* in1, T* out, T c, size_t n) {
  if (mv.v == 1) return launch_one<T, FN, HAS_IN1, 1, 4>(L, mv.persist, nc, in0, in1, out, c, n);
  if (mv.v == 4) return launch_one<T, FN, HAS_IN1, 4, 4>(L, mv.persist, nc, in0, in1, out, c, n);
  if (mv.u == 2) return launch_one<T, FN, HAS_IN1, 8, 2>(L, mv.persist, nc, in0, in1, out, c, n);
  return launch_one<T, FN, HAS_IN1, 8, 4>(L, mv.persist, nc, in0, in1, out, c, n);
}

template <typename T>
cudaError_t launch_t(const Launch& L, const MapVariant& mv, int fn, bool has_in1, T c, const T* in0, const T* in1,
                     T* out, size_t n) {
  const bool nc = (static_cast<const void*>(in0) != out) && (static_cast<const void*>(in1) != out);
#define SKEL_MAP_CASE(F)                                                                      \
  case F:                                                                                     \
    return has_in1 ? launch_vu<T, F, true>(L, mv, nc, in0, in1, out, c, n)                    \
                   : launch_vu<T, F, false>(L, mv, nc, in0, in1, out, c, n);
  switch (fn) {
    SKEL_MAP_CASE(FN_ADD)
    SKEL_MAP_CASE(FN_MULT)
    SKEL_MAP_CASE(FN_MAX)
    case FN_SAXPY:
      return launch_vu<T, FN_SAXPY, true>(L, mv, nc, in0, in1, out, c, n);
  }
#undef SKEL_MAP_CASE
  return cudaErrorInvalidValue;
}

template <typename T, int V, int U>
cudaError_t launch_map3_one(const Launch& L, bool persist, bool nc, const T* in0, const T* in1, const T* in2, T* out, size_t n) {
  constexpr size_t TILE = size_t(MAP_THREADS) * V * U;
  size_t ntiles = (n + TILE - 1) / TILE;
  size_t grid = persist ? (size_t)L.sms * 8 : ntiles;
  if (grid > ntiles) grid = ntiles;
  if (grid > 0x7fffffffu) grid = 0x7fffffffu;
  if (nc) map3_kernel<T, V, U, true><<<(unsigned)grid, MAP_THREADS, 0, L.stream>>>(in0, in1, in2, out, n);
  else map3_kernel<T, V, U, false><<<(unsigned)grid, MAP_THREADS, 0, L.stream>>>(in0, in1, in2, out, n);
  ++*L.launches;
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_map3_t(const Launch& L, const MapVariant& mv, const T* in0, const T* in1, const T* in2, T* out, size_t n) {
  const void* o = out;
  const bool nc = in0 != o && in1 != o && in2 != o;
  if (mv.v == 1) return launch_map3_one<T, 1, 4>(L, mv.persist, nc, in0, in1, in2, out, n);
  if (mv.v == 4) return launch_map3_one<T, 4, 2>(L, mv.persist, nc, in0, in1, in2, out, n);
  return launch_map3_one<T, 8, 2>(L, mv.persist, nc, in0, in1, in2, out, n);
}

}  // namespace

cudaError_t launch_map3(const Launch& L, int v, int dtype, const void* in0, const void* in1, const void* in2, void* out,
                        size_t n) {
  if (n == 0) return cudaSuccess;
  const MapVariant& mv = kMapVariants[v];
  if (dtype == DT_F32)
    return launch_map3_t<float>(L, mv, static_cast<const float*>(in0), static_cast<const float*>(in1),
                                static_cast<const float*>(in2), static_cast<float*>(out), n);
  return launch_map3_t<int32_t>(L, mv, static_cast<const int32_t*>(in0), static_cast<const int32_t*>(in1),
                                static_cast<const int32_t*>(in2), static_cast<int32_t*>(out), n);
}

int map_variant_count() { return kNumMapVariants; }
const char* map_variant_name(int v) { return (v >= 0 && v < kNumMapVariants) ? kMapVariants[v].name : nullptr; }

bool map_variant_ok(int v, const void* in0, const void* in1, const void* out, size_t) {
  if (v < 0 || v >= kNumMapVariants) return false;
  const size_t a = size_t(kMapVariants[v].v) * 4;
  return aligned_to(in0, a) && aligned_to(in1, a) && aligned_to(out, a);
}

cudaError_t launch_map(const Launch& L, int v, int dtype, int fn, bool has_in1, uint32_t cbits, const void* in0,
                       const void* in1, void* out, size_t n) {
  if (n == 0) return cudaSuccess;
  const MapVariant& mv = kMapVariants[v];
  if (dtype == DT_F32) {
    float c;
    memcpy(&c, &cbits, 4);
    return launch_t<float>(L, mv, fn, has_in1, c, static_cast<const float*>(in0), static_cast<const float*>(in1),
                           static_cast<float*>(out), n);
  }
  return launch_t<int32_t>(L, mv, fn, has_in1, static_cast<int32_t>(cbits), static_cast<const int32_t*>(in0),
                           static_cast<const int32_t*>(in1), static_cast<int32_t*>(out), n);
}

}  // namespace skel
