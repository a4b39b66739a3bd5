// MapOverlap 2D skeleton and the column-wise 1D form on a matrix (readings 5 and 6):
//   out[i][j] = sum_{a=-ry..ry} sum_{b=-rx..rx} W[a+ry][b+rx] * X~[i+a][j+b]
// X~ = pad (CONSTANT), X[clamp i][clamp j] (DUPLICATE, every index clamped on its own) or
// X[i mod rows][j mod cols] (CYCLIC).
// Column-wise 1D is the rx = 0 case (a (2r+1) x 1 filter).
//
// Variants:
//  * "direct": any radii, any alignment; one output per thread, neighbours served by L1/L2.
//  * "tiled_oy{4,8}": a (8*OY + 2ry) x (128 + 2*ceil4(rx)) tile is staged in shared memory with
//    128-bit loads; a thread produces a 4 (x) by OY (y) block of outputs. Each staged row it reads
//    (one or a few 128-bit shared loads) is reused for up to 2ry+1 output rows from registers;
//    weights come from the constant bank; all taps are unrolled (radii are template parameters).
// Summation order: a outer, b inner, like the definition. When a filter has more than 33 taps,
// each filter row is summed on its own and the row sums are then added (rounding-error bound
// (2rx+1 + 2ry) * 2^-24 of sum|W x| instead of (2ry+1)(2rx+1) * 2^-24).
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

// ---- direct --------------------------------------------------------------------------------
// Filter rows are summed separately in chains of at most 17 taps, then added.
template <typename WT>
__global__ void __launch_bounds__(256)
overlap2d_direct_kernel(const __grid_constant__ WT W, int ry, int rx, int edge, float pad, const float* in, float* out,
                        size_t rows, size_t cols) {
  const size_t total = rows * cols;
  const int fw = 2 * rx + 1;
  for (size_t idx = blockIdx.x * size_t(blockDim.x) + threadIdx.x; idx < total; idx += size_t(gridDim.x) * blockDim.x) {
    const long long i = static_cast<long long>(idx / cols);
    const long long j = static_cast<long long>(idx - size_t(i) * cols);
    const bool interior = i - ry >= 0 && i + ry < (long long)rows && j - rx >= 0 && j + rx < (long long)cols;
    float acc = 0.f;
    if (rx == 0) {  // column-wise 1D: chains of 16 taps
      for (int a0 = 0; a0 <= 2 * ry; a0 += 16) {
        const int a1 = min(a0 + 16, 2 * ry + 1);
        float p = 0.f;
        for (int a = a0; a < a1; ++a) {
          const float v = interior ? __ldg(in + (i + a - ry) * (long long)cols + j)
                                   : ext2(in, rows, cols, i + a - ry, j, edge, pad);
          p = fmaf(W.w[a], v, p);
        }
        acc = a0 == 0 ? p : acc + p;
      }
    } else {
      for (int a = 0; a <= 2 * ry; ++a) {
        float p = 0.f;
        for (int b = 0; b <= 2 * rx; ++b) {
          const float v = interior ? __ldg(in + (i + a - ry) * (long long)cols + (j + b - rx))
                                   : ext2(in, rows, cols, i + a - ry, j + b - rx, edge, pad);
          p = fmaf(W.w[a * fw + b], v, p);
        }
        acc = a == 0 ? p : acc + p;
      }
    }
    out[idx] = acc;
  }
}

// ---- shared-memory tiled, register blocked -------------------------------------------------
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

// a thread's 4 (x) by OY (y) outputs from the staged tile, written to `out`
// PK: taps whose window index is even use one FFMA2 per output pair (the pair (v[i], v[i+1]) of a
// 128-bit shared load is an aligned register pair); odd taps stay scalar. Each output still sums its
// taps in the order b = 0 .. 2RX, so the result is bit-identical to the scalar form.
template <int RY, int RX, int OY, typename WT, bool PK = false>
__device__ __forceinline__ void compute_tile2(const float* sm, const WT& W, float* out, long long rows, long long cols,
                                              long long r0, long long c0) {
  constexpr int RXP = (RX + 3) / 4 * 4;
  constexpr int SW = T2_TW + 2 * RXP;
  constexpr int NGX = (4 + 2 * RXP) / 4;
  constexpr int FW = 2 * RX + 1;
  constexpr bool PER_ROW = (2 * RY + 1) * (2 * RX + 1) > 33;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  float acc[OY][4];
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
        if constexpr (PER_ROW) {
          float p[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int b = 0; b < FW; ++b) {
            if (PK && (RXP - RX + b) % 2 == 0) {
              fma2_into(p[0], p[1], W.w[a * FW + b], v[RXP - RX + b], v[RXP - RX + b + 1]);
              fma2_into(p[2], p[3], W.w[a * FW + b], v[RXP - RX + b + 2], v[RXP - RX + b + 3]);
            } else {
#pragma unroll
              for (int e = 0; e < 4; ++e) p[e] = fmaf(W.w[a * FW + b], v[RXP - RX + b + e], p[e]);
            }
          }
#pragma unroll
          for (int e = 0; e < 4; ++e) acc[o][e] = a == 0 ? p[e] : acc[o][e] + p[e];
        } else {
#pragma unroll
          for (int b = 0; b < FW; ++b) {
            if (PK && (RXP - RX + b) % 2 == 0) {
              fma2_into(acc[o][0], acc[o][1], W.w[a * FW + b], v[RXP - RX + b], v[RXP - RX + b + 1]);
              fma2_into(acc[o][2], acc[o][3], W.w[a * FW + b], v[RXP - RX + b + 2], v[RXP - RX + b + 3]);
            } else {
#pragma unroll
              for (int e = 0; e < 4; ++e) acc[o][e] = fmaf(W.w[a * FW + b], v[RXP - RX + b + e], acc[o][e]);
            }
          }
        }
      }
    }
  }
  const long long oc = c0 + tx * 4;
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
    compute_tile2<RY, RX, OY, WT>(sm, W, out, rows, cols, r0, c0);
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

template <typename WT>
cudaError_t launch_direct2(const Launch& L, const WT& w, int ry, int rx, int edge, float pad, const float* in,
                           float* out, size_t rows, size_t cols) {
  const size_t total = rows * cols;
  size_t grid = (total + 255) / 256;
  const size_t cap = size_t(L.sms) * 64;
  if (grid > cap) grid = cap;
  overlap2d_direct_kernel<WT><<<(unsigned)grid, 256, 0, L.stream>>>(w, ry, rx, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

const char* const kNames[] = {"direct", "tiled_oy4", "tiled_oy8", "tiled_oy4_db", "tiled_oy8_db", "tiled_oy4_db_ffma2",
                              "tiled_oy8_db_ffma2"};
constexpr int kNumVariants = 7;

inline bool tiled_alignment_ok(const void* in, const void* out, size_t cols) {
  return reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0 && cols % 4 == 0;
}

}  // namespace

// ---- column-wise 1D ----------------------------------------------------------------------------
int overlap1d_col_variant_count() { return kNumVariants; }
const char* overlap1d_col_variant_name(int v) { return (v >= 0 && v < kNumVariants) ? kNames[v] : nullptr; }
bool overlap1d_col_variant_ok(int v, int r, const void* in, const void* out, size_t, size_t cols) {
  if (v < 0 || v >= kNumVariants) return false;
  if (v == 0) return true;
  const bool templated = r == 1 || r == 2 || r == 3 || r == 4 || r == 8 || r == 16;
  return templated && tiled_alignment_ok(in, out, cols);
}

cudaError_t launch_overlap1d_cols(const Launch& L, int v, const Weights1D& w, int r, int edge, float pad,
                                  const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  if (v == 0) return launch_direct2<Weights1D>(L, w, r, 0, edge, pad, in, out, rows, cols);
#define SKEL_COL_CASE(R)                                                                                      \
  case R:                                                                                                     \
    switch (v) {                                                                                              \
      case 1: return launch_tiled2<R, 0, 4, Weights1D>(L, w, edge, pad, in, out, rows, cols);                 \
      case 2: return launch_tiled2<R, 0, 8, Weights1D>(L, w, edge, pad, in, out, rows, cols);                 \
      case 3: return launch_tiled2_db<R, 0, 4, Weights1D>(L, w, edge, pad, in, out, rows, cols);              \
      case 4: return launch_tiled2_db<R, 0, 8, Weights1D>(L, w, edge, pad, in, out, rows, cols);              \
      case 5: return launch_tiled2_db<R, 0, 4, Weights1D, true>(L, w, edge, pad, in, out, rows, cols);        \
      case 6: return launch_tiled2_db<R, 0, 8, Weights1D, true>(L, w, edge, pad, in, out, rows, cols);        \
    }                                                                                                         \
    break;
  switch (r) {
    SKEL_COL_CASE(1)
    SKEL_COL_CASE(2)
    SKEL_COL_CASE(3)
    SKEL_COL_CASE(4)
    SKEL_COL_CASE(8)
    SKEL_COL_CASE(16)
  }
#undef SKEL_COL_CASE
  return cudaErrorInvalidValue;
}

// ---- 2D ----------------------------------------------------------------------------------------
int overlap2d_variant_count() { return kNumVariants; }
const char* overlap2d_variant_name(int v) { return (v >= 0 && v < kNumVariants) ? kNames[v] : nullptr; }
bool overlap2d_variant_ok(int v, int ry, int rx, const void* in, const void* out, size_t, size_t cols) {
  if (v < 0 || v >= kNumVariants) return false;
  if (v == 0) return true;
  const bool templated = ry == rx && ry >= 1 && ry <= 4;
  return templated && tiled_alignment_ok(in, out, cols);
}

cudaError_t launch_overlap2d(const Launch& L, int v, const Weights2D& w, int ry, int rx, int edge, float pad,
                             const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  if (v == 0) return launch_direct2<Weights2D>(L, w, ry, rx, edge, pad, in, out, rows, cols);
#define SKEL_2D_CASE(R)                                                                                       \
  case R:                                                                                                     \
    switch (v) {                                                                                              \
      case 1: return launch_tiled2<R, R, 4, Weights2D>(L, w, edge, pad, in, out, rows, cols);                 \
      case 2: return launch_tiled2<R, R, 8, Weights2D>(L, w, edge, pad, in, out, rows, cols);                 \
      case 3: return launch_tiled2_db<R, R, 4, Weights2D>(L, w, edge, pad, in, out, rows, cols);              \
      case 4: return launch_tiled2_db<R, R, 8, Weights2D>(L, w, edge, pad, in, out, rows, cols);              \
      case 5: return launch_tiled2_db<R, R, 4, Weights2D, true>(L, w, edge, pad, in, out, rows, cols);        \
      case 6: return launch_tiled2_db<R, R, 8, Weights2D, true>(L, w, edge, pad, in, out, rows, cols);        \
    }                                                                                                         \
    break;
  switch (ry) {
    SKEL_2D_CASE(1)
    SKEL_2D_CASE(2)
    SKEL_2D_CASE(3)
    SKEL_2D_CASE(4)
  }
#undef SKEL_2D_CASE
  return cudaErrorInvalidValue;
}

}  // namespace skel
