// Cross-call fusion of a chain of dependent skeleton calls on one vector (the
// GPU-only analogue of PAPER.md L137/L149: optimise over a chain of calls instead of call by call):
//
//     [ Map(f, c):  A' = f(A, c) ]   ->   MapOverlap1D(w, r, edge):  B = stencil(A')   ->   [ Reduce(op):  s = (+) B ]
//
// ONE kernel reads A once, writes A' (if the Map is part of the chain) and B, and folds B into the
// reduction on the fly: 12 B/elem instead of 8 + 8 + 4 = 20 for the three separate calls. Every
// element is computed by the same arithmetic as in the separate kernels (Map: one rounding of f;
// MapOverlap: taps accumulated in ascending order with FMAs; Reduce: fixed-order trees, no float
// atomics), so the results stay inside the tolerances of the separate calls.
//
// Structure = the register-window MapOverlap variant (overlap1d.cu "regshfl_o16"): a thread owns 16
// consecutive elements (two 256-bit loads), applies the Map in registers, gets the r halo values of
// each side from the neighbouring lanes by shuffles (lanes 0 and 31 read and map them from memory),
// and keeps 4 reduction accumulators. `map_out` must not alias `in`: the halo of a warp is read
// from `in` while another block may already have stored its part of A' (api.cu gives an in-place
// Map a fresh buffer and swaps it into the container).
#include "common.cuh"
#include "kernels.hpp"
#include <string.h>

namespace skel {
namespace {

enum : int { EDGE_CONSTANT = 0, EDGE_DUPLICATE = 1, EDGE_CYCLIC = 2 };
constexpr int FU_THREADS = 256;
constexpr int OP_NONE = -1;

template <int MAPF> __device__ __forceinline__ float map1(float c, float a) {
  if constexpr (MAPF == FN_IDENT) return a;
  else return apply_fn<MAPF>(c, a, c);
}

// A'~[j]: the mapped vector seen through the edge policy (CONSTANT pads with `pad`, NOT with f(pad))
template <int MAPF>
__device__ __forceinline__ float ext_mapped(const float* x, long long n, long long j, int edge, float pad, float c) {
  if (j >= 0 && j < n) return map1<MAPF>(c, __ldg(x + j));
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) {
    long long m = j % n;
    return map1<MAPF>(c, __ldg(x + (m < 0 ? m + n : m)));
  }
  return map1<MAPF>(c, __ldg(x + (j < 0 ? 0 : n - 1)));
}

__device__ __forceinline__ void fma2_into(float& lo, float& hi, float w, float x0, float x1) {
  unsigned long long ww, xx, cc, d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ww) : "f"(w), "f"(w));
  asm("mov.b64 %0, {%1, %2};" : "=l"(xx) : "f"(x0), "f"(x1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(cc) : "f"(lo), "f"(hi));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(ww), "l"(xx), "l"(cc));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}

template <int R, int MAPF, int OP>
__global__ void __launch_bounds__(FU_THREADS)
fused_chain_kernel(const __grid_constant__ Weights1D W, int edge, float pad, float c, const float* in, float* map_out,
                   float* ov_out, size_t n, unsigned long long* tagged, unsigned* ticket, uint32_t epoch, float* result) {
  constexpr int O = 16;
  constexpr int TILE = FU_THREADS * O;
  constexpr int ROP = OP == OP_NONE ? FN_ADD : OP;  // only instantiates the helpers; unused when OP_NONE
  static_assert(R >= 1 && R <= O, "halo comes from the direct neighbours only");
  __shared__ float smem[32];
  __shared__ unsigned s_order;
  // tagged end (common.cuh): the ticket is drawn when the block STARTS; its latency hides under the loads
  unsigned order = 0;
  if constexpr (OP != OP_NONE) {
    if (threadIdx.x == 0 && gridDim.x > 1) order = atomicInc(ticket + 4, gridDim.x - 1);  // wraps to 0: self-resetting
  }
  const int lane = threadIdx.x & 31;
  const long long ln = static_cast<long long>(n);
  const size_t ntiles = (n + TILE - 1) / TILE;
  float red[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) red[q] = identity<float, ROP>();

  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long long c0 = static_cast<long long>(tile * TILE) + threadIdx.x * O;
    float win[O + 2 * R];
    const bool full = c0 + O <= ln;
    if (full) {
      uint32_t a[8], b[8];
      ld_stream<8, true>(a, in + c0);
      ld_stream<8, true>(b, in + c0 + 8);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        win[R + j] = map1<MAPF>(c, __uint_as_float(a[j]));
        win[R + 8 + j] = map1<MAPF>(c, __uint_as_float(b[j]));
      }
      if constexpr (MAPF != FN_IDENT) {
        uint32_t m0[8], m1[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) { m0[j] = __float_as_uint(win[R + j]); m1[j] = __float_as_uint(win[R + 8 + j]); }
        st_stream<8>(map_out + c0, m0);
        st_stream<8>(map_out + c0 + 8, m1);
      }
    } else {
#pragma unroll
      for (int j = 0; j < O; ++j) {
        win[R + j] = ext_mapped<MAPF>(in, ln, c0 + j, edge, pad, c);
        if constexpr (MAPF != FN_IDENT)
          if (c0 + j < ln) map_out[c0 + j] = win[R + j];
      }
    }
#pragma unroll
    for (int j = 0; j < R; ++j) {
      const float l = __shfl_up_sync(0xffffffffu, win[R + O - R + j], 1);
      const float r = __shfl_down_sync(0xffffffffu, win[R + j], 1);
      win[j] = l;
      win[R + O + j] = r;
    }
    if (lane == 0) {
#pragma unroll
      for (int j = 0; j < R; ++j) win[j] = ext_mapped<MAPF>(in, ln, c0 - R + j, edge, pad, c);
    }
    if (lane == 31) {
#pragma unroll
      for (int j = 0; j < R; ++j) win[R + O + j] = ext_mapped<MAPF>(in, ln, c0 + O + j, edge, pad, c);
    }
    float acc[O];
#pragma unroll
    for (int o = 0; o < O; ++o) acc[o] = 0.f;
    constexpr bool PK = R >= 8;  // as in overlap1d_shfl_kernel: bit-identical to the scalar chain
#pragma unroll
    for (int k = 0; k <= 2 * R; ++k) {
      if (PK && (k + R) % 2 == 0) {
#pragma unroll
        for (int o = 0; o < O; o += 2) fma2_into(acc[o], acc[o + 1], W.w[k], win[o + k], win[o + k + 1]);
      } else {
#pragma unroll
        for (int o = 0; o < O; ++o) acc[o] = fmaf(W.w[k], win[o + k], acc[o]);
      }
    }
    if (full) {
      uint32_t r0[8], r1[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) { r0[e] = __float_as_uint(acc[e]); r1[e] = __float_as_uint(acc[8 + e]); }
      st_stream<8>(ov_out + c0, r0);
      st_stream<8>(ov_out + c0 + 8, r1);
      if constexpr (OP != OP_NONE) {
#pragma unroll
        for (int o = 0; o < O; ++o) red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], acc[o]);
      }
    } else {
#pragma unroll
      for (int o = 0; o < O; ++o)
        if (c0 + o < ln) {
          ov_out[c0 + o] = acc[o];
          if constexpr (OP != OP_NONE) red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], acc[o]);
        }
    }
  }

  if constexpr (OP != OP_NONE) {
    float v = apply_fn<ROP>(0.f, apply_fn<ROP>(0.f, red[0], red[1]), apply_fn<ROP>(0.f, red[2], red[3]));
    v = block_reduce<float, ROP>(v, smem);
    if (gridDim.x == 1) {
      if (threadIdx.x == 0) *result = v;
      return;
    }
    if (threadIdx.x == 0) {  // partial and launch number in ONE 64-bit store: no fence, nothing to wait for
      const unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned long long)to_bits(v);
      asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(tagged + blockIdx.x), "l"(w) : "memory");
      s_order = order;
    }
    __syncthreads();
    // the 8 blocks that started last fold the slots in a fixed order (run-to-run deterministic; common.cuh)
    const unsigned ord = s_order;
    if (ord + TAG_P >= gridDim.x) fold_tagged<float, ROP, FU_THREADS>(tagged, gridDim.x, ord, epoch, result, smem);
  }
}

// The same chain in the "regshfl_2x8" layout (overlap1d.cu): a warp owns 512 consecutive elements, lane l the two
// 8-element chunks A = [8l, 8l+8) and B = [256+8l, 256+8l+8), so every 256-bit load and store of a warp covers 1024
// contiguous bytes (whole 128-byte lines) instead of every other 32-byte sector of 2048 bytes. Halos by wrap-around
// shuffles (lane 31's chunk A borders lane 0's chunk B). r <= 8. Same arithmetic per element as fused_chain_kernel.
template <int R, int MAPF, int OP>
__global__ void __launch_bounds__(FU_THREADS)
fused_chain2_kernel(const __grid_constant__ Weights1D W, int edge, float pad, float c, const float* in, float* map_out,
                    float* ov_out, size_t n, unsigned long long* tagged, unsigned* ticket, uint32_t epoch, float* result) {
  constexpr int C = 8, TILE = FU_THREADS * 2 * C;
  constexpr int ROP = OP == OP_NONE ? FN_ADD : OP;
  static_assert(R >= 1 && R <= C, "halo comes from the direct neighbours only");
  constexpr unsigned FULLM = 0xffffffffu;
  __shared__ float smem[32];
  __shared__ unsigned s_order;
  // tagged end (common.cuh): the ticket is drawn when the block STARTS; its latency hides under the loads
  unsigned order = 0;
  if constexpr (OP != OP_NONE) {
    if (threadIdx.x == 0 && gridDim.x > 1) order = atomicInc(ticket + 4, gridDim.x - 1);  // wraps to 0: self-resetting
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long ln = static_cast<long long>(n);
  const size_t ntiles = (n + TILE - 1) / TILE;
  float red[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) red[q] = identity<float, ROP>();

  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long long wbase = static_cast<long long>(tile * TILE) + warp * (64 * C);
    const long long cA = wbase + C * lane, cB = cA + 32 * C;
    const bool full = wbase + 64 * C <= ln;  // warp-uniform
    float wa[C + 2 * R], wb[C + 2 * R];
    if (full) {
      uint32_t a[8], b[8];
      ld_stream<8, true>(a, in + cA);
      ld_stream<8, true>(b, in + cB);
#pragma unroll
      for (int j = 0; j < C; ++j) {
        wa[R + j] = map1<MAPF>(c, __uint_as_float(a[j]));
        wb[R + j] = map1<MAPF>(c, __uint_as_float(b[j]));
      }
      if constexpr (MAPF != FN_IDENT) {
        uint32_t m0[8], m1[8];
#pragma unroll
        for (int j = 0; j < C; ++j) { m0[j] = __float_as_uint(wa[R + j]); m1[j] = __float_as_uint(wb[R + j]); }
        st_stream<8>(map_out + cA, m0);
        st_stream<8>(map_out + cB, m1);
      }
    } else {
#pragma unroll
      for (int j = 0; j < C; ++j) {
        wa[R + j] = ext_mapped<MAPF>(in, ln, cA + j, edge, pad, c);
        wb[R + j] = ext_mapped<MAPF>(in, ln, cB + j, edge, pad, c);
        if constexpr (MAPF != FN_IDENT) {
          if (cA + j < ln) map_out[cA + j] = wa[R + j];
          if (cB + j < ln) map_out[cB + j] = wb[R + j];
        }
      }
    }
    const int prev = (lane + 31) & 31, next = (lane + 1) & 31;
#pragma unroll
    for (int j = 0; j < R; ++j) {
      const float tA = __shfl_sync(FULLM, wa[C + j], prev);
      const float hA = __shfl_sync(FULLM, wa[R + j], next);
      const float tB = __shfl_sync(FULLM, wb[C + j], prev);
      const float hB = __shfl_sync(FULLM, wb[R + j], next);
      wa[j] = tA;
      wa[R + C + j] = lane == 31 ? hB : hA;
      wb[j] = lane == 0 ? tA : tB;
      wb[R + C + j] = hB;
    }
    if (lane == 0) {
#pragma unroll
      for (int j = 0; j < R; ++j) wa[j] = ext_mapped<MAPF>(in, ln, cA - R + j, edge, pad, c);
    }
    if (lane == 31) {
#pragma unroll
      for (int j = 0; j < R; ++j) wb[R + C + j] = ext_mapped<MAPF>(in, ln, cB + C + j, edge, pad, c);
    }
    float accA[C], accB[C];
#pragma unroll
    for (int o = 0; o < C; ++o) accA[o] = accB[o] = 0.f;
    constexpr bool PK = R >= 8;
#pragma unroll
    for (int k = 0; k <= 2 * R; ++k) {
      if (PK && (k + R) % 2 == 0) {
#pragma unroll
        for (int o = 0; o < C; o += 2) {
          fma2_into(accA[o], accA[o + 1], W.w[k], wa[o + k], wa[o + k + 1]);
          fma2_into(accB[o], accB[o + 1], W.w[k], wb[o + k], wb[o + k + 1]);
        }
      } else {
#pragma unroll
        for (int o = 0; o < C; ++o) {
          accA[o] = fmaf(W.w[k], wa[o + k], accA[o]);
          accB[o] = fmaf(W.w[k], wb[o + k], accB[o]);
        }
      }
    }
    if (full) {
      uint32_t r0[8], r1[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) { r0[e] = __float_as_uint(accA[e]); r1[e] = __float_as_uint(accB[e]); }
      st_stream<8>(ov_out + cA, r0);
      st_stream<8>(ov_out + cB, r1);
      if constexpr (OP != OP_NONE) {
#pragma unroll
        for (int o = 0; o < C; ++o) {
          red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], accA[o]);
          red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], accB[o]);
        }
      }
    } else {
#pragma unroll
      for (int o = 0; o < C; ++o) {
        if (cA + o < ln) {
          ov_out[cA + o] = accA[o];
          if constexpr (OP != OP_NONE) red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], accA[o]);
        }
        if (cB + o < ln) {
          ov_out[cB + o] = accB[o];
          if constexpr (OP != OP_NONE) red[o & 3] = apply_fn<ROP>(0.f, red[o & 3], accB[o]);
        }
      }
    }
  }

  if constexpr (OP != OP_NONE) {
    float v = apply_fn<ROP>(0.f, apply_fn<ROP>(0.f, red[0], red[1]), apply_fn<ROP>(0.f, red[2], red[3]));
    v = block_reduce<float, ROP>(v, smem);
    if (gridDim.x == 1) {
      if (threadIdx.x == 0) *result = v;
      return;
    }
    if (threadIdx.x == 0) {  // partial and launch number in ONE 64-bit store: no fence, nothing to wait for
      const unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned long long)to_bits(v);
      asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(tagged + blockIdx.x), "l"(w) : "memory");
      s_order = order;
    }
    __syncthreads();
    // the 8 blocks that started last fold the slots in a fixed order (run-to-run deterministic; common.cuh)
    const unsigned ord = s_order;
    if (ord + TAG_P >= gridDim.x) fold_tagged<float, ROP, FU_THREADS>(tagged, gridDim.x, ord, epoch, result, smem);
  }
}

template <int R, int MAPF, int OP>
cudaError_t launch_rmo(const Launch& L, const Scratch& S, const Weights1D& w, int edge, float pad, float c,
                       const float* in, float* map_out, float* ov_out, size_t n, float* result) {
  constexpr size_t TILE = size_t(FU_THREADS) * 16;
  size_t grid = (n + TILE - 1) / TILE;
  if (OP != OP_NONE && grid > MAX_PARTIALS) grid = MAX_PARTIALS;
  if (grid > 0x7fffffffu) grid = 0x7fffffffu;
  if (OP != OP_NONE && ++S.red_epoch == 0) {  // 2^32 launches: start over from cleared slots (reduce.cu)
    cudaError_t e = cudaMemsetAsync(S.red_tagged, 0, size_t(MAX_PARTIALS + 8) * 8, L.stream);
    if (e != cudaSuccess) return e;
    S.red_epoch = 1;
  }
  if constexpr (R <= 8)  // warp-contiguous layout (fewer halo shuffles than loads saved only up to r = 8)
    fused_chain2_kernel<R, MAPF, OP><<<(unsigned)grid, FU_THREADS, 0, L.stream>>>(
        w, edge, pad, c, in, map_out, ov_out, n, S.red_tagged, S.ticket, S.red_epoch, result);
  else
    fused_chain_kernel<R, MAPF, OP><<<(unsigned)grid, FU_THREADS, 0, L.stream>>>(
        w, edge, pad, c, in, map_out, ov_out, n, S.red_tagged, S.ticket, S.red_epoch, result);
  ++*L.launches;
  return cudaGetLastError();
}

template <int R, int MAPF>
cudaError_t launch_rm(const Launch& L, const Scratch& S, int red_op, const Weights1D& w, int edge, float pad, float c,
                      const float* in, float* map_out, float* ov_out, size_t n, float* result) {
  switch (red_op) {
    case OP_NONE: return launch_rmo<R, MAPF, OP_NONE>(L, S, w, edge, pad, c, in, map_out, ov_out, n, result);
    case FN_ADD: return launch_rmo<R, MAPF, FN_ADD>(L, S, w, edge, pad, c, in, map_out, ov_out, n, result);
    case FN_MAX: return launch_rmo<R, MAPF, FN_MAX>(L, S, w, edge, pad, c, in, map_out, ov_out, n, result);
  }
  return cudaErrorInvalidValue;
}

template <int R>
cudaError_t launch_r(const Launch& L, const Scratch& S, int map_fn, int red_op, const Weights1D& w, int edge, float pad,
                     float c, const float* in, float* map_out, float* ov_out, size_t n, float* result) {
  switch (map_fn) {
    case FN_IDENT: return launch_rm<R, FN_IDENT>(L, S, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case FN_ADD: return launch_rm<R, FN_ADD>(L, S, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case FN_MULT: return launch_rm<R, FN_MULT>(L, S, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case FN_MAX: return launch_rm<R, FN_MAX>(L, S, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
  }
  return cudaErrorInvalidValue;
}

inline bool al32(const void* p) { return reinterpret_cast<uintptr_t>(p) % 32 == 0; }

}  // namespace

bool fused_chain_ok(int map_fn, int r, int red_op, const void* in, const void* map_out, const void* ov_out, size_t n) {
  // radii between the instantiated ones run zero-padded (kernels.hpp); beyond r = 8 the register-window form loses
  // to the separate TMA-fed MapOverlap kernel (225 against 210 us per iteration at r = 16, n = 2^26): not fused
  const bool rt = r >= 0 && r <= 8;
  const bool mf = map_fn == FN_IDENT || map_fn == FN_ADD || map_fn == FN_MULT || map_fn == FN_MAX;
  const bool ro = red_op == FUSED_NO_REDUCE || red_op == FN_ADD || red_op == FN_MAX;
  if (!rt || !mf || !ro || n == 0) return false;
  if (map_fn == FN_IDENT && red_op == FUSED_NO_REDUCE) return false;  // a lone MapOverlap is not a chain
  if (!al32(in) || !al32(ov_out) || (map_fn != FN_IDENT && !al32(map_out))) return false;
  if (in == ov_out || (map_fn != FN_IDENT && (map_out == in || map_out == ov_out))) return false;
  return true;
}

cudaError_t launch_fused_chain(const Launch& L, const Scratch& S, int map_fn, uint32_t cbits, const Weights1D& w, int r,
                               int edge, float pad, int red_op, const float* in, float* map_out, float* ov_out, size_t n,
                               float* result) {
  float c;
  memcpy(&c, &cbits, 4);
  if (const int R = padded_radius_1d(r); R != r) {
    if (R < 0) return cudaErrorInvalidValue;
    return launch_fused_chain(L, S, map_fn, cbits, pad_weights_1d(w, r, R), R, edge, pad, red_op, in, map_out, ov_out, n, result);
  }
  switch (r) {
    case 1: return launch_r<1>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case 2: return launch_r<2>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case 3: return launch_r<3>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case 4: return launch_r<4>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case 8: return launch_r<8>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
    case 16: return launch_r<16>(L, S, map_fn, red_op, w, edge, pad, c, in, map_out, ov_out, n, result);
  }
  return cudaErrorInvalidValue;
}

}  // namespace skel
