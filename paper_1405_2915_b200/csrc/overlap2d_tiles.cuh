// Shared-memory tiled kernels of MapOverlap 2D and of the column-wise 1D form (rx = 0), templated on
// the radii. Included by overlap2d_inst.cu, which is compiled once per radius (one translation unit
// per instantiation set keeps the build parallel); overlap2d.cu holds the direct kernel and the
// dispatch.
//
//  * "tiled_oy{4,8}": one block per tile. A (8*OY + 2ry) x (128 + 2*ceil4(rx)) window is staged in
//    shared memory with 128-bit loads; a thread produces a 4 (x) by OY (y) block of outputs. Each
//    staged row it reads is reused for up to 2ry+1 output rows from registers; weights come from the
//    constant bank / uniform registers; all taps are unrolled.
//  * "tiled_oy{4,8}_db": persistent blocks, two shared-memory buffers filled by cp.async.
//  * "tma_oy{4,8}": persistent blocks, 2 or 3 shared-memory buffers filled by ONE 2-D tensor copy per
//    tile (TMA, cp.async.bulk.tensor: out-of-range cells arrive as zeros), full/empty mbarriers
//    instead of block barriers, tile coordinates advanced without divisions. Tiles whose window
//    leaves the matrix are patched in shared memory with the edge policy before they are used.
// FFMA2 (the persistent 2D variants): taps whose window index is even use one fma.rn.f32x2 per output pair (the pair
// (v[i], v[i+1]) of a 128-bit shared load is an aligned register pair); odd taps stay scalar. Each
// output still sums its taps in the order b = 0 .. 2RX: bit-identical to the scalar form.
// "tma_bx*" (broadcast form, RX > 0): EVERY tap is an FFMA2 whatever its alignment. The pair of outputs (2q, 2q+1) of a
// thread receives window element x[j] with the taps d = j - 2q (output 2q) and d - 1 (output 2q+1): one FFMA2 whose
// data operand is the single register x[j] broadcast to both halves (SASS: FFMA2 R, R.F32, UR.F32x2, R) and whose
// weight operand is the pair (w[d], w[d-1]) held in a uniform-register pair (host-built table WPairs2D, constant bank).
// The first and last tap of a filter row have no partner and stay scalar: 2RX FFMA2 + 2 FFMA per output pair and
// filter row (9x9: 10 instructions for 18 FMAs instead of 13), no wasted FMA lane. Every output still receives its
// taps in ascending order, one fused multiply-add each: bit-identical to the scalar form. "bx2": a thread owns two
// 4-wide strips 128 columns apart (tile 32 x 256, two TMA boxes per stage), so a weight pair loaded into uniform
// registers feeds twice as many FFMA2.
// Summation order: a outer, b inner, like the definition. When a filter has more than 33 taps,
// each filter row is summed on its own and the row sums are then added.
#pragma once
#include <cuda.h>
#include "common.cuh"
#include "kernels.hpp"

namespace skel {
namespace {

enum : int { EDGE_CONSTANT = 0, EDGE_DUPLICATE = 1, EDGE_CYCLIC = 2 };

__device__ __forceinline__ float ext2(const float* X, long long rows, long long cols, long long p, long long q,
                                      int edge, float pad) {
  if (p >= 0 && p < rows && q >= 0 && q < cols) return __ldg(X + p * cols + q);
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) {  // each index wraps on its own (non-negative remainder)
    p %= rows;
    q %= cols;
    p = p < 0 ? p + rows : p;
    q = q < 0 ? q + cols : q;
  } else {
    p = p < 0 ? 0 : (p >= rows ? rows - 1 : p);
    q = q < 0 ? 0 : (q >= cols ? cols - 1 : q);
  }
  return __ldg(X + p * cols + q);
}

constexpr int T2_THREADS = 256;  // 32 (x) by 8 (y)
constexpr int T2_TW = 128;       // tile width in outputs: 32 threads x 4

// stage X~[r0-RY .. r0+TH+RY) x [c0-RXP .. c0+TW+RXP) into `sm` (SH rows of SW floats).
// ASYNC: groups that lie inside the matrix go through cp.async (LDGSTS, no registers, completion
// via cp.async.wait_group); groups touching an edge are computed with the edge policy and stored.
template <int RY, int RX, int OY, bool ASYNC>
__device__ __forceinline__ void stage_tile2(float* sm, const float* in, long long rows, long long cols, long long r0,
                                            long long c0, int edge, float pad) {
  constexpr int RXP = (RX + 3) / 4 * 4;
  constexpr int TH = 8 * OY, SW = T2_TW + 2 * RXP, SH = TH + 2 * RY;
#pragma unroll 4
  for (int g = threadIdx.x; g < SH * (SW / 4); g += T2_THREADS) {
    const int gy = g / (SW / 4), gx = g - gy * (SW / 4);
    const long long p = r0 - RY + gy, q = c0 - RXP + 4 * gx;
    float* dst = sm + gy * SW + 4 * gx;
    if (p >= 0 && p < rows && q >= 0 && q + 3 < cols) {
      if constexpr (ASYNC) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(in + p * cols + q) : "memory");
      } else {
        uint32_t raw[4];
        ld_stream<4, true>(raw, in + p * cols + q);
        *reinterpret_cast<float4*>(dst) =
            make_float4(__uint_as_float(raw[0]), __uint_as_float(raw[1]), __uint_as_float(raw[2]), __uint_as_float(raw[3]));
      }
    } else {
      float4 v;
      v.x = ext2(in, rows, cols, p, q, edge, pad);
      v.y = ext2(in, rows, cols, p, q + 1, edge, pad);
      v.z = ext2(in, rows, cols, p, q + 2, edge, pad);
      v.w = ext2(in, rows, cols, p, q + 3, edge, pad);
      *reinterpret_cast<float4*>(dst) = v;
    }
  }
}

// packed fp32 pairs (Blackwell FFMA2): d = a * b + c on both halves of an aligned register pair
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void fma2_into(float& lo, float& hi, float w, float x0, float x1) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pack2(w, w)), "l"(pack2(x0, x1)), "l"(pack2(lo, hi)));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}

// geometry of a staged tile (per strip: an SH x SW window, one TMA box)
template <int RY, int RX, int OY, int XS = 1> struct Tile2Geom {
  static constexpr int RXP = (RX + 3) / 4 * 4;
  static constexpr int TH = 8 * OY, SW = T2_TW + 2 * RXP, SH = TH + 2 * RY;
  static constexpr int TW = T2_TW * XS;                        // tile width in outputs: XS strips of 128 columns
  static constexpr unsigned BOX_BYTES = unsigned(SH) * SW * 4u;  // one TMA box (one strip's window)
  static constexpr unsigned BOX_STRIDE = XS == 1 ? BOX_BYTES : (BOX_BYTES + 127u) / 128u * 128u;  // TMA wants 128-byte aligned boxes
  static constexpr unsigned STAGE_BYTES = BOX_BYTES * XS;      // bytes the TMA copies deliver per stage
  static constexpr unsigned STAGE_STRIDE = (BOX_STRIDE * XS + 127u) / 128u * 128u;
};

// weight pairs of the broadcast form: p[a][d] = (w[a][d], w[a][d-1]) for d = 0 .. FW (w[a][-1] = w[a][FW] = 0);
// rows padded to a multiple of 16 bytes so that one LDCU.128 fetches two pairs
template <int RY, int RX> struct alignas(16) WPairs2D {
  static constexpr int FW = 2 * RX + 1, NP = (FW + 2) / 2 * 2;
  float2 p[2 * RY + 1][NP];
};
template <int RY, int RX> inline void make_wpairs(WPairs2D<RY, RX>& P, const float* w /* (2RY+1) x (2RX+1) */) {
  constexpr int FW = 2 * RX + 1;
  for (int a = 0; a <= 2 * RY; ++a)
    for (int d = 0; d < WPairs2D<RY, RX>::NP; ++d) {
      P.p[a][d].x = d < FW ? w[a * FW + d] : 0.f;
      P.p[a][d].y = (d >= 1 && d <= FW) ? w[a * FW + d - 1] : 0.f;
    }
}
// (lo, hi) += (wp.x, wp.y) * (x, x): the data register is broadcast, the weight pair comes from uniform registers
__device__ __forceinline__ void fma2_bcast(float& lo, float& hi, float2 wp, float x) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pack2(x, x)), "l"(pack2(wp.x, wp.y)), "l"(pack2(lo, hi)));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}

// Broadcast form of compute_tile2: a thread's XS strips of 4 (x) by OY (y) outputs; strip s is staged in its own
// SH x SW window at sm + s * SH * SW and covers output columns c0 + 128 s + 4 tx .. + 3.
template <int RY, int RX, int OY, int XS>
__device__ __forceinline__ void compute_tile2_bx(const float* sm, const WPairs2D<RY, RX>& P, float* out, long long rows,
                                                 long long cols, long long r0, long long c0, bool full_tile) {
  constexpr int RXP = (RX + 3) / 4 * 4;
  constexpr int SW = T2_TW + 2 * RXP;
  constexpr int NGX = (4 + 2 * RXP) / 4;
  constexpr int FW = 2 * RX + 1, OFF = RXP - RX;
  constexpr bool GROUPED = (2 * RY + 1) * FW > 33;
  constexpr int GR = GROUPED ? (33 / FW > 0 ? 33 / FW : 1) : 2 * RY + 1;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  float acc[XS][OY][4];
  float part[XS][GROUPED ? OY : 1][4];
#pragma unroll
  for (int s = 0; s < XS; ++s)
#pragma unroll
    for (int o = 0; o < OY; ++o)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[s][o][e] = 0.f;

#pragma unroll
  for (int ir = 0; ir < OY + 2 * RY; ++ir) {
    float v[XS][4 * NGX];
#pragma unroll
    for (int s = 0; s < XS; ++s) {
      const float* srow = sm + s * int(Tile2Geom<RY, RX, OY, XS>::BOX_STRIDE / 4) + (ty * OY + ir) * SW + tx * 4;
#pragma unroll
      for (int g = 0; g < NGX; ++g) {
        const float4 t = *reinterpret_cast<const float4*>(srow + 4 * g);
        v[s][4 * g] = t.x; v[s][4 * g + 1] = t.y; v[s][4 * g + 2] = t.z; v[s][4 * g + 3] = t.w;
      }
    }
#pragma unroll
    for (int o = 0; o < OY; ++o) {
      const int a = ir - o;
      if (a >= 0 && a <= 2 * RY) {
        if (GROUPED && a % GR == 0) {
#pragma unroll
          for (int s = 0; s < XS; ++s)
#pragma unroll
            for (int e = 0; e < 4; ++e) part[s][GROUPED ? o : 0][e] = 0.f;
        }
#pragma unroll
        for (int d = 0; d <= FW; ++d) {
          const float2 wp = P.p[a][d];
#pragma unroll
          for (int s = 0; s < XS; ++s) {
            float* dstp = GROUPED ? part[s][GROUPED ? o : 0] : acc[s][o];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
              const float x = v[s][OFF + d + 2 * q];
              if (d == 0) dstp[2 * q] = fmaf(wp.x, x, dstp[2 * q]);
              else if (d == FW) dstp[2 * q + 1] = fmaf(wp.y, x, dstp[2 * q + 1]);
              else fma2_bcast(dstp[2 * q], dstp[2 * q + 1], wp, x);
            }
          }
        }
        if (GROUPED && (a % GR == GR - 1 || a == 2 * RY)) {
#pragma unroll
          for (int s = 0; s < XS; ++s)
#pragma unroll
            for (int e = 0; e < 4; ++e)
              acc[s][o][e] = a < GR ? part[s][GROUPED ? o : 0][e] : acc[s][o][e] + part[s][GROUPED ? o : 0][e];
        }
      }
    }
  }
#pragma unroll
  for (int s = 0; s < XS; ++s) {
    const long long oc = c0 + s * T2_TW + tx * 4;
    if (full_tile) {
      float* dst = out + (r0 + ty * OY) * cols + oc;
#pragma unroll
      for (int o = 0; o < OY; ++o, dst += cols) {
        uint32_t raw[4] = {__float_as_uint(acc[s][o][0]), __float_as_uint(acc[s][o][1]), __float_as_uint(acc[s][o][2]),
                           __float_as_uint(acc[s][o][3])};
        st_stream<4>(dst, raw);
      }
    } else {
#pragma unroll
      for (int o = 0; o < OY; ++o) {
        const long long orow = r0 + ty * OY + o;
        if (orow < rows) {
          float* dst = out + orow * cols + oc;
          if (oc + 3 < cols) {
            uint32_t raw[4] = {__float_as_uint(acc[s][o][0]), __float_as_uint(acc[s][o][1]), __float_as_uint(acc[s][o][2]),
                               __float_as_uint(acc[s][o][3])};
            st_stream<4>(dst, raw);
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (oc + e < cols) dst[e] = acc[s][o][e];
          }
        }
      }
    }
  }
}

// a thread's 4 (x) by OY (y) outputs from the staged tile, written to `out`.
// full_tile = the caller knows that the whole tile lies inside the matrix: the row and column checks
// vanish and the output address is advanced by `cols` per row.
template <int RY, int RX, int OY, typename WT, bool PK_, typename T = float>
__device__ __forceinline__ void compute_tile2(const float* sm, const WT& W, float* out, long long rows, long long cols,
                                              long long r0, long long c0, bool full_tile = false) {
  constexpr bool PK = PK_ && StencilOps<T>::kFloat;
  constexpr int RXP = (RX + 3) / 4 * 4;
  constexpr int SW = T2_TW + 2 * RXP;
  constexpr int NGX = (4 + 2 * RXP) / 4;
  constexpr int FW = 2 * RX + 1;
  // Filters with more than 33 taps are summed in groups of GR whole filter rows (at most 33 taps per
  // chain, e.g. 9x9: three chains of 27), and the group sums are added: rounding-error bound
  // (GR * FW + #groups - 1) * 2^-24 of sum|W x| (9x9: 29 * 2^-24 = 1.73e-6), DESIGN.md "Tolerances".
  constexpr bool GROUPED = (2 * RY + 1) * FW > 33;
  constexpr int GR = GROUPED ? (33 / FW > 0 ? 33 / FW : 1) : 2 * RY + 1;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  float acc[OY][4];
  float part[GROUPED ? OY : 1][4];  // running sum of the current group of filter rows, per output row
#pragma unroll
  for (int o = 0; o < OY; ++o)
#pragma unroll
    for (int e = 0; e < 4; ++e) acc[o][e] = 0.f;

#pragma unroll
  for (int ir = 0; ir < OY + 2 * RY; ++ir) {
    const float* srow = sm + (ty * OY + ir) * SW + tx * 4;
    float v[4 * NGX];
#pragma unroll
    for (int g = 0; g < NGX; ++g) {
      const float4 t = *reinterpret_cast<const float4*>(srow + 4 * g);
      v[4 * g] = t.x; v[4 * g + 1] = t.y; v[4 * g + 2] = t.z; v[4 * g + 3] = t.w;
    }
#pragma unroll
    for (int o = 0; o < OY; ++o) {
      const int a = ir - o;  // filter row that this staged row feeds for output row o
      if (a >= 0 && a <= 2 * RY) {
        float* dstp = GROUPED ? part[GROUPED ? o : 0] : acc[o];
        if (GROUPED && a % GR == 0) {
#pragma unroll
          for (int e = 0; e < 4; ++e) dstp[e] = 0.f;
        }
#pragma unroll
        for (int b = 0; b < FW; ++b) {
          if (PK && (RXP - RX + b) % 2 == 0) {
            fma2_into(dstp[0], dstp[1], W.w[a * FW + b], v[RXP - RX + b], v[RXP - RX + b + 1]);
            fma2_into(dstp[2], dstp[3], W.w[a * FW + b], v[RXP - RX + b + 2], v[RXP - RX + b + 3]);
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) dstp[e] = StencilOps<T>::mad(W.w[a * FW + b], v[RXP - RX + b + e], dstp[e]);
          }
        }
        if (GROUPED && (a % GR == GR - 1 || a == 2 * RY)) {  // the group is complete
#pragma unroll
          for (int e = 0; e < 4; ++e) acc[o][e] = a < GR ? dstp[e] : StencilOps<T>::add(acc[o][e], dstp[e]);
        }
      }
    }
  }
  const long long oc = c0 + tx * 4;
  if (full_tile) {
    float* dst = out + (r0 + ty * OY) * cols + oc;
#pragma unroll
    for (int o = 0; o < OY; ++o, dst += cols) {
      uint32_t raw[4] = {__float_as_uint(acc[o][0]), __float_as_uint(acc[o][1]), __float_as_uint(acc[o][2]),
                         __float_as_uint(acc[o][3])};
      st_stream<4>(dst, raw);
    }
  } else {
#pragma unroll
    for (int o = 0; o < OY; ++o) {
      const long long orow = r0 + ty * OY + o;
      if (orow < rows) {
        float* dst = out + orow * cols + oc;
        if (oc + 3 < cols) {
          uint32_t raw[4] = {__float_as_uint(acc[o][0]), __float_as_uint(acc[o][1]), __float_as_uint(acc[o][2]),
                             __float_as_uint(acc[o][3])};
          st_stream<4>(dst, raw);
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (oc + e < cols) dst[e] = acc[o][e];
        }
      }
    }
  }
}

template <int RY, int RX, int OY, typename WT>
__global__ void __launch_bounds__(T2_THREADS)
overlap2d_tiled_kernel(const __grid_constant__ WT W, int edge, float pad, const float* in, float* out, size_t rows,
                       size_t cols) {
  constexpr int TH = 8 * OY;
  extern __shared__ __align__(16) float sm[];
  const size_t tiles_x = (cols + T2_TW - 1) / T2_TW, tiles_y = (rows + TH - 1) / TH;
  const size_t ntiles = tiles_x * tiles_y;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t tyi = tile / tiles_x;
    const long long r0 = static_cast<long long>(tyi * TH);
    const long long c0 = static_cast<long long>((tile - tyi * tiles_x) * T2_TW);
    stage_tile2<RY, RX, OY, false>(sm, in, rows, cols, r0, c0, edge, pad);
    __syncthreads();
    compute_tile2<RY, RX, OY, WT, false>(sm, W, out, rows, cols, r0, c0);
    __syncthreads();
  }
}

// Double-buffered persistent form ("_db"): a grid of co-resident blocks walks the tiles; while a
// block computes tile i from one shared-memory buffer, the cp.async copies of tile i+1 fill the
// other, so the load phase of a block no longer alternates with its compute phase.
template <int RY, int RX, int OY, typename WT, bool PK>
__global__ void __launch_bounds__(T2_THREADS)
overlap2d_tiled_db_kernel(const __grid_constant__ WT W, int edge, float pad, const float* in, float* out, size_t rows,
                          size_t cols) {
  constexpr int RXP = (RX + 3) / 4 * 4;
  constexpr int TH = 8 * OY, SW = T2_TW + 2 * RXP, SH = TH + 2 * RY;
  extern __shared__ __align__(16) float sm[];
  const size_t tiles_x = (cols + T2_TW - 1) / T2_TW, tiles_y = (rows + TH - 1) / TH;
  const size_t ntiles = tiles_x * tiles_y;
  auto origin = [&](size_t tile, long long& r0, long long& c0) {
    const size_t tyi = tile / tiles_x;
    r0 = static_cast<long long>(tyi * TH);
    c0 = static_cast<long long>((tile - tyi * tiles_x) * T2_TW);
  };
  // Interior tiles (staged window fully inside the matrix) take a fast path: the shared-memory and
  // global offsets of this thread's 128-bit groups do not depend on the tile, so they are computed
  // once and every group costs one address add + one cp.async. Border tiles use stage_tile2.
  constexpr int GROUPS = SH * (SW / 4), NG = (GROUPS + T2_THREADS - 1) / T2_THREADS;
  int soff[NG], goff[NG];
#pragma unroll
  for (int k = 0; k < NG; ++k) {
    const int g = threadIdx.x + k * T2_THREADS;
    const int gy = g / (SW / 4), gx = g - gy * (SW / 4);
    soff[k] = g < GROUPS ? (gy * SW + 4 * gx) * 4 : -1;  // byte offset in the buffer
    goff[k] = (gy - RY) * static_cast<int>(cols) + 4 * gx - RXP;  // element offset from the tile origin
  }
  const bool small_pitch = cols * size_t(SH) < (size_t(1) << 30);
  auto stage = [&](float* dstbuf, long long tr0, long long tc0) {
    const bool interior = small_pitch && tr0 - RY >= 0 && tr0 + TH + RY <= static_cast<long long>(rows) &&
                          tc0 - RXP >= 0 && tc0 + T2_TW + RXP <= static_cast<long long>(cols);
    if (interior) {
      const float* src = in + tr0 * static_cast<long long>(cols) + tc0;
      const uint32_t dbase = smem_u32(dstbuf);
#pragma unroll
      for (int k = 0; k < NG; ++k)
        if (soff[k] >= 0)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dbase + soff[k]), "l"(src + goff[k]) : "memory");
    } else {
      stage_tile2<RY, RX, OY, true>(dstbuf, in, rows, cols, tr0, tc0, edge, pad);
    }
  };
  long long r0, c0;
  size_t tile = blockIdx.x;
  if (tile >= ntiles) return;
  origin(tile, r0, c0);
  stage(sm, r0, c0);
  asm volatile("cp.async.commit_group;" ::: "memory");
  int buf = 0;
  for (; tile < ntiles; tile += gridDim.x, buf ^= 1) {
    const size_t next = tile + gridDim.x;
    if (next < ntiles) {
      long long nr0, nc0;
      origin(next, nr0, nc0);
      stage(sm + (buf ^ 1) * SH * SW, nr0, nc0);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 1;" ::: "memory");  // the current tile has landed (this thread's copies)
    __syncthreads();                                       // ... and everybody else's
    origin(tile, r0, c0);
    compute_tile2<RY, RX, OY, WT, PK>(sm + buf * SH * SW, W, out, rows, cols, r0, c0);
    __syncthreads();  // the buffer is refilled by the next iteration's prefetch
  }
}

// ---- TMA-fed persistent form ("tma_*") -----------------------------------------------------------
// G = 148 x occupancy co-resident blocks take tiles from a global counter (dynamic assignment: with a static
// b, b+G, ... walk the blocks of an SM drift apart - the warp scheduler favours the oldest warps - and the SM ends the
// kernel with one or two of its blocks already gone; ncu showed 2.1 of 3 blocks resident on average). Thread 0 is the
// producer: it fetches the next tile id (atomicAdd; the counter is never reset, the host passes its value at launch as
// `tile_base` and advances its own copy by ntiles: ntiles - G successful fetches + one failing fetch per block), writes the tile's origin into
// the stage's `coord` slot and issues one cp.async.bulk.tensor.2d per strip that copies the (SH x SW) window into
// stage (it + STAGES-1) % STAGES and completes on that stage's `full` mbarrier; cells outside the matrix arrive as
// zeros. Every thread waits on `full`, reads `coord`, computes, and each warp arrives on the stage's `empty` mbarrier
// when it has finished reading; thread 0 waits on `empty` before it refills the stage. A stage whose `coord` is
// negative ends the walk. There is no block barrier on the interior path, so the 8 warps of a block drift by up to
// STAGES-1 tiles.
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(smem_dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar))
      : "memory");
}


// XS > 1 / BX: the broadcast form (compute_tile2_bx; WT = WPairs2D<RY, RX>), XS TMA boxes per stage.
template <int RY, int RX, int OY, typename WT, bool PK, int STAGES, int XS = 1, bool BX = false, int MINB = 0,
          typename T = float>
__global__ void __launch_bounds__(T2_THREADS, MINB)
overlap2d_tma_kernel(const __grid_constant__ WT W, const __grid_constant__ CUtensorMap tmap, int edge, float pad,
                     const float* in, float* out, int rows, int cols, int tiles_x, int ntiles, unsigned* tile_ctr,
                     unsigned tile_base) {
  using G = Tile2Geom<RY, RX, OY, XS>;
  constexpr int RXP = G::RXP, TH = G::TH, SW = G::SW, SH = G::SH, TW = G::TW;
  extern __shared__ __align__(128) unsigned char smraw[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw + STAGES * G::STAGE_STRIDE);
  uint64_t* empty = full + STAGES;
  int2* coord = reinterpret_cast<int2*>(empty + STAGES);  // (r0, c0) of the tile in each stage; r0 < 0: no more tiles
  auto stage_ptr = [&](int s) { return reinterpret_cast<float*>(smraw + s * G::STAGE_STRIDE); };
  const int lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, T2_THREADS / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();
  // thread 0: the first tile is the block's own index, later ids come from the counter (+ gridDim.x); the fetch of tile
  // k+1 is issued while tile k is requested and examined one iteration later, so its latency overlaps a tile's compute.
  // The id that ends the walk is examined before any further fetch: exactly one failing fetch per block.
  unsigned t_next = blockIdx.x;
  bool exhausted = false;
  auto produce = [&](int s) {  // thread 0: next tile into stage s, or mark the stage as the end of the walk
    const unsigned t = t_next;
    if (!exhausted) exhausted = t >= unsigned(ntiles);
    if (!exhausted) t_next = atomicAdd(tile_ctr, 1u) - tile_base + gridDim.x;
    if (!exhausted) {
      const int y = int(t) / tiles_x, x = int(t) - y * tiles_x;
      coord[s] = make_int2(y * TH, x * TW);
      mbar_arrive_expect_tx(full + s, G::STAGE_BYTES);
#pragma unroll
      for (int k = 0; k < XS; ++k)
        tma_load_2d(reinterpret_cast<unsigned char*>(stage_ptr(s)) + k * G::BOX_STRIDE, &tmap, x * TW + k * T2_TW - RXP,
                    y * TH - RY, full + s);
    } else {
      coord[s] = make_int2(-1, 0);
      mbar_arrive(full + s);
    }
  };
  if (threadIdx.x == 0) {
#pragma unroll
    for (int d = 0; d < STAGES - 1; ++d) produce(d);
  }
  // zeros are what CONSTANT with pad = 0 wants; any other policy patches the cells outside the matrix
  const bool patch_needed = !(edge == EDGE_CONSTANT && bits_are_zero(pad));
  int s = 0, ph = 0;           // stage and parity of this iteration's `full` wait
  int tgt = STAGES - 1, tph = 1;  // thread 0: stage to refill and parity of its `empty` wait
  for (int it = 0;; ++it) {
    if (threadIdx.x == 0) {
      if (it > 0) mbar_wait(empty + tgt, tph);  // every warp has finished reading tile it-1
      produce(tgt);
    }
    tgt = tgt + 1 == STAGES ? 0 : tgt + 1;
    if (tgt == 0) tph ^= 1;
    mbar_wait(full + s, ph);
    const int2 rc = coord[s];
    if (rc.x < 0) break;
    const int r0 = rc.x, c0 = rc.y;
    float* sm = stage_ptr(s);
    const bool window_inside = r0 - RY >= 0 && r0 + TH + RY <= rows && c0 - RXP >= 0 && c0 + TW + RXP <= cols;
    if (!window_inside && patch_needed) {  // block-uniform branch
      for (int idx = threadIdx.x; idx < XS * SH * SW; idx += T2_THREADS) {
        const int k = idx / (SH * SW), rem = idx - k * (SH * SW);
        const int gy = rem / SW, gx = rem - gy * SW;
        const int p = r0 - RY + gy, q = c0 + k * T2_TW - RXP + gx;
        if (p < 0 || p >= rows || q < 0 || q >= cols) sm[k * int(G::BOX_STRIDE / 4) + rem] = ext2(in, rows, cols, p, q, edge, pad);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic writes before the next TMA refill
      __syncthreads();
    }
    if constexpr (BX)
      compute_tile2_bx<RY, RX, OY, XS>(sm, W, out, rows, cols, r0, c0, r0 + TH <= rows && c0 + TW <= cols);
    else
      compute_tile2<RY, RX, OY, WT, PK, T>(sm, W, out, rows, cols, r0, c0, r0 + TH <= rows && c0 + T2_TW <= cols);
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + s);
    s = s + 1 == STAGES ? 0 : s + 1;
    if (s == 0) ph ^= 1;
  }
}

template <int RY, int RX, int OY> constexpr size_t tiled2_smem() {
  return size_t(8 * OY + 2 * RY) * (T2_TW + 2 * ((RX + 3) / 4 * 4)) * sizeof(float);
}

template <int RY, int RX, int OY, typename WT>
cudaError_t launch_tiled2(const Launch& L, const WT& w, int edge, float pad, const float* in, float* out, size_t rows,
                          size_t cols) {
  constexpr size_t smem = tiled2_smem<RY, RX, OY>();
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(overlap2d_tiled_kernel<RY, RX, OY, WT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_done = true;
  }
  const size_t ntiles = ((cols + T2_TW - 1) / T2_TW) * ((rows + 8 * OY - 1) / (8 * OY));
  const size_t grid = ntiles < 0x7fffffffu ? ntiles : 0x7fffffffu;
  overlap2d_tiled_kernel<RY, RX, OY, WT><<<(unsigned)grid, T2_THREADS, smem, L.stream>>>(w, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

template <int RY, int RX, int OY, typename WT, bool PK = false>
cudaError_t launch_tiled2_db(const Launch& L, const WT& w, int edge, float pad, const float* in, float* out, size_t rows,
                             size_t cols) {
  constexpr size_t smem = 2 * tiled2_smem<RY, RX, OY>();
  auto kern = overlap2d_tiled_db_kernel<RY, RX, OY, WT, PK>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T2_THREADS, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  const size_t ntiles = ((cols + T2_TW - 1) / T2_TW) * ((rows + 8 * OY - 1) / (8 * OY));
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T2_THREADS, smem, L.stream>>>(w, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

// L2 promotion 64 B: a window row starts 16 bytes before a 512-byte boundary; with 128- or 256-byte promotion the
// over-fetch at both ends of every row reached HBM (ncu: DRAM reads 1.08 / 1.13 x the matrix, 1.05 x with 64 B).
// Tensor map of the input matrix with a (box_w x box_h) box (host side; the driver entry point is
// looked up once through the runtime, libcuda is not linked). The last map is cached: chained calls
// on the same container re-use it.
inline cudaError_t make_tmap_2d(CUtensorMap* out, const float* base, size_t rows, size_t cols, int box_w, int box_h) {
  using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    encode = reinterpret_cast<EncodeFn>(fn);
  }
  struct Key { const float* base; size_t rows, cols; int bw, bh; };
  static thread_local Key last = {nullptr, 0, 0, 0, 0};  // per host thread: contexts may live on different threads
  static thread_local CUtensorMap last_map;
  if (last.base == base && last.rows == rows && last.cols == cols && last.bw == box_w && last.bh == box_h) {
    *out = last_map;
    return cudaSuccess;
  }
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * sizeof(float)};
  const cuuint32_t box[2] = {cuuint32_t(box_w), cuuint32_t(box_h)};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  last = {base, rows, cols, box_w, box_h};
  last_map = *out;
  return cudaSuccess;
}

template <int RY, int RX, int OY, typename WT, bool PK, int STAGES, typename T = float>
cudaError_t launch_tma2(const Launch& L, const WT& w, int edge, float pad, const float* in, float* out, size_t rows,
                        size_t cols) {
  using G = Tile2Geom<RY, RX, OY>;
  constexpr size_t smem = size_t(STAGES) * G::STAGE_STRIDE + 3 * STAGES * sizeof(uint64_t);  // stages, full/empty, coord
  static_assert(smem <= 227 * 1024, "stages do not fit");
  auto kern = overlap2d_tma_kernel<RY, RX, OY, WT, PK, STAGES, 1, false, 0, T>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T2_THREADS, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tmap;
  cudaError_t e = make_tmap_2d(&tmap, in, rows, cols, G::SW, G::SH);
  if (e != cudaSuccess) return e;
  const size_t tiles_x = (cols + T2_TW - 1) / T2_TW;
  const size_t ntiles = tiles_x * ((rows + G::TH - 1) / G::TH);
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T2_THREADS, smem, L.stream>>>(w, tmap, edge, pad, in, out, (int)rows, (int)cols, (int)tiles_x,
                                                        (int)ntiles, L.tile_ctr, *L.tile_next);
  *L.tile_next += unsigned(ntiles);  // ntiles - grid tiles are fetched from the counter, every block fetches one id past the end
  ++*L.launches;
  return cudaGetLastError();
}

// broadcast form (RX > 0): the weight-pair table is built here, per call
template <int RY, int RX, int OY, int XS, int STAGES, int MINB>
cudaError_t launch_tma2_bx(const Launch& L, const Weights2D& w, int edge, float pad, const float* in, float* out,
                           size_t rows, size_t cols) {
  using G = Tile2Geom<RY, RX, OY, XS>;
  using WP = WPairs2D<RY, RX>;
  constexpr size_t smem = size_t(STAGES) * G::STAGE_STRIDE + 3 * STAGES * sizeof(uint64_t);  // stages, full/empty, coord
  static_assert(smem <= 227 * 1024, "stages do not fit");
  auto kern = overlap2d_tma_kernel<RY, RX, OY, WP, false, STAGES, XS, true, MINB>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T2_THREADS, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tmap;
  cudaError_t e = make_tmap_2d(&tmap, in, rows, cols, G::SW, G::SH);
  if (e != cudaSuccess) return e;
  WP P;
  make_wpairs<RY, RX>(P, w.w);
  const size_t tiles_x = (cols + G::TW - 1) / G::TW;
  const size_t ntiles = tiles_x * ((rows + G::TH - 1) / G::TH);
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T2_THREADS, smem, L.stream>>>(P, tmap, edge, pad, in, out, (int)rows, (int)cols, (int)tiles_x,
                                                        (int)ntiles, L.tile_ctr, *L.tile_next);
  *L.tile_next += unsigned(ntiles);
  ++*L.launches;
  return cudaGetLastError();
}

// every tiled variant of one (RY, RX) pair; v = variant id of overlap2d.cu's table (v >= 1)
template <int RY, int RX, typename WT>
cudaError_t launch_tiled_any(const Launch& L, int v, int dtype, const WT& w, int edge, float pad, const float* in,
                             float* out, size_t rows, size_t cols) {
  constexpr bool PK = RX > 0;  // FFMA2 pays when a row feeds several taps; the column form has one tap per row
  if (dtype != DT_F32) {  // int32 elements: the TMA-fed variants (scalar multiply-add modulo 2^32)
    switch (v) {
      case 5: return launch_tma2<RY, RX, 4, WT, false, 3, int32_t>(L, w, edge, pad, in, out, rows, cols);
      case 6: return launch_tma2<RY, RX, 8, WT, false, RX == 0 ? 3 : 2, int32_t>(L, w, edge, pad, in, out, rows, cols);
      case 7: return launch_tma2<RY, RX, 4, WT, false, 2, int32_t>(L, w, edge, pad, in, out, rows, cols);
    }
    return cudaErrorInvalidValue;
  }
  switch (v) {
    case 1: return launch_tiled2<RY, RX, 4, WT>(L, w, edge, pad, in, out, rows, cols);
    case 2: return launch_tiled2<RY, RX, 8, WT>(L, w, edge, pad, in, out, rows, cols);
    case 3: return launch_tiled2_db<RY, RX, 4, WT, PK>(L, w, edge, pad, in, out, rows, cols);
    case 4: return launch_tiled2_db<RY, RX, 8, WT, PK>(L, w, edge, pad, in, out, rows, cols);
    case 5: return launch_tma2<RY, RX, 4, WT, PK, 3>(L, w, edge, pad, in, out, rows, cols);
    case 6: return launch_tma2<RY, RX, 8, WT, PK, RX == 0 ? 3 : 2>(L, w, edge, pad, in, out, rows, cols);
    case 7: return launch_tma2<RY, RX, 4, WT, PK, 2>(L, w, edge, pad, in, out, rows, cols);  // 2 stages: 5 resident blocks
  }
  if constexpr (RX > 0) {  // broadcast-FFMA2 forms (dense 2D only)
    switch (v) {
      case 8: return launch_tma2_bx<RY, RX, 4, 1, 3, 3>(L, w, edge, pad, in, out, rows, cols);
      case 9: return launch_tma2_bx<RY, RX, 4, 1, 2, 1>(L, w, edge, pad, in, out, rows, cols);
      case 10: return launch_tma2_bx<RY, RX, 4, 2, 2, 2>(L, w, edge, pad, in, out, rows, cols);
      case 11: return launch_tma2_bx<RY, RX, 2, 2, 3, 3>(L, w, edge, pad, in, out, rows, cols);
    }
  }
  return cudaErrorInvalidValue;
}

}  // namespace
}  // namespace skel
