// MapOverlap 2D skeleton and the column-wise 1D form on a matrix (readings 5 and 6):
//   out[i][j] = sum_{a=-ry..ry} sum_{b=-rx..rx} W[a+ry][b+rx] * X~[i+a][j+b]
// X~ = pad (CONSTANT), X[clamp i][clamp j] (DUPLICATE, every index clamped on its own) or
// X[i mod rows][j mod cols] (CYCLIC).
// Column-wise 1D is the rx = 0 case (a (2r+1) x 1 filter).
//
// This file: the "direct" variant (any radii, any alignment; one output per thread, neighbours
// served by L1/L2), the variant table and the dispatch. The shared-memory tiled variants live in
// overlap2d_tiles.cuh and are instantiated per radius in overlap2d_inst.cu.
#include "overlap2d_tiles.cuh"  // ext2, the edge-policy enum

namespace skel {
namespace {

// ---- direct --------------------------------------------------------------------------------
// Filter rows are summed separately in chains of at most 17 taps, then added.
template <typename WT, typename T>
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
    if (rx == 0) {  // column-wise 1D: one chain up to 33 taps (like the tiled variants), else chains of 16 taps
      const int chain = 2 * ry + 1 <= 33 ? 33 : 16;
      for (int a0 = 0; a0 <= 2 * ry; a0 += chain) {
        const int a1 = min(a0 + chain, 2 * ry + 1);
        float p = 0.f;
        for (int a = a0; a < a1; ++a) {
          const float v = interior ? __ldg(in + (i + a - ry) * (long long)cols + j)
                                   : ext2(in, rows, cols, i + a - ry, j, edge, pad);
          p = StencilOps<T>::mad(W.w[a], v, p);
        }
        acc = a0 == 0 ? p : StencilOps<T>::add(acc, p);
      }
    } else {
      for (int a = 0; a <= 2 * ry; ++a) {
        float p = 0.f;
        for (int b = 0; b <= 2 * rx; ++b) {
          const float v = interior ? __ldg(in + (i + a - ry) * (long long)cols + (j + b - rx))
                                   : ext2(in, rows, cols, i + a - ry, j + b - rx, edge, pad);
          p = StencilOps<T>::mad(W.w[a * fw + b], v, p);
        }
        acc = a == 0 ? p : StencilOps<T>::add(acc, p);
      }
    }
    out[idx] = acc;
  }
}

template <typename WT>
cudaError_t launch_direct2(const Launch& L, int dtype, const WT& w, int ry, int rx, int edge, float pad, const float* in,
                           float* out, size_t rows, size_t cols) {
  const size_t total = rows * cols;
  size_t grid = (total + 255) / 256;
  const size_t cap = size_t(L.sms) * 64;
  if (grid > cap) grid = cap;
  if (dtype == DT_F32)
    overlap2d_direct_kernel<WT, float><<<(unsigned)grid, 256, 0, L.stream>>>(w, ry, rx, edge, pad, in, out, rows, cols);
  else
    overlap2d_direct_kernel<WT, int32_t><<<(unsigned)grid, 256, 0, L.stream>>>(w, ry, rx, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

// 8..11: the broadcast-FFMA2 forms of the TMA kernel (overlap2d_tiles.cuh "tma_bx*"), dense 2D only
const char* const kNames[] = {"direct", "tiled_oy4", "tiled_oy8", "tiled_oy4_db", "tiled_oy8_db",
                              "tma_oy4", "tma_oy8", "tma_oy4_s2", "tma_bx_oy4", "tma_bx_oy4_s2", "tma_bx2_oy4_s2",
                              "tma_bx2_oy2"};
constexpr int kNumVariants = 12;
constexpr int kNumColVariants = 8;

inline bool tiled_alignment_ok(const void* in, const void* out, size_t rows, size_t cols) {
  return reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0 && cols % 4 == 0 &&
         rows < (size_t(1) << 30) && cols < (size_t(1) << 30) && ((rows + 31) / 32) * ((cols + 127) / 128) < (size_t(1) << 30);
}

}  // namespace

// ---- column-wise 1D ----------------------------------------------------------------------------
int overlap1d_col_variant_count() { return kNumColVariants; }
const char* overlap1d_col_variant_name(int v) { return (v >= 0 && v < kNumColVariants) ? kNames[v] : nullptr; }
bool overlap1d_col_variant_ok(int v, int dtype, int r, const void* in, const void* out, size_t rows, size_t cols) {
  if (v < 0 || v >= kNumColVariants) return false;
  if (v == 0) return true;
  if (dtype != DT_F32 && (v < 5 || v > 7)) return false;  // i32: direct and the TMA-fed variants
  return r >= 0 && r <= 16 && tiled_alignment_ok(in, out, rows, cols);  // other radii run zero-padded (kernels.hpp)
}

cudaError_t launch_overlap1d_cols(const Launch& L, int v, int dtype, const Weights1D& w, int r, int edge, float pad,
                                  const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  if (v == 0) return launch_direct2<Weights1D>(L, dtype, w, r, 0, edge, pad, in, out, rows, cols);
  if (const int R = padded_radius_1d(r); R != r) {
    if (R < 0) return cudaErrorInvalidValue;
    return launch_overlap1d_cols(L, v, dtype, pad_weights_1d(w, r, R), R, edge, pad, in, out, rows, cols);
  }
  switch (r) {
    case 1: return launch_overlap1d_cols_tiled<1>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 2: return launch_overlap1d_cols_tiled<2>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 3: return launch_overlap1d_cols_tiled<3>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 4: return launch_overlap1d_cols_tiled<4>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 8: return launch_overlap1d_cols_tiled<8>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 16: return launch_overlap1d_cols_tiled<16>(L, v, dtype, w, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

// ---- 2D ----------------------------------------------------------------------------------------
int overlap2d_variant_count() { return kNumVariants; }
const char* overlap2d_variant_name(int v) { return (v >= 0 && v < kNumVariants) ? kNames[v] : nullptr; }
bool overlap2d_variant_ok(int v, int dtype, int ry, int rx, const void* in, const void* out, size_t rows, size_t cols) {
  if (v < 0 || v >= kNumVariants) return false;
  if (v == 0) return true;
  if (dtype != DT_F32 && (v < 5 || v > 7)) return false;  // i32: direct and the TMA-fed variants
  // rectangular filters and ry = rx = 0 run the square filter of radius max(ry, rx, 1) zero-padded (kernels.hpp)
  return ry >= 0 && rx >= 0 && ry <= 4 && rx <= 4 && tiled_alignment_ok(in, out, rows, cols);
}

cudaError_t launch_overlap2d(const Launch& L, int v, int dtype, const Weights2D& w, int ry, int rx, int edge, float pad,
                             const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  if (v == 0) return launch_direct2<Weights2D>(L, dtype, w, ry, rx, edge, pad, in, out, rows, cols);
  if (ry != rx || ry < 1) {
    const int R = ry > rx ? ry : (rx > 1 ? rx : 1);
    if (R > 4) return cudaErrorInvalidValue;
    return launch_overlap2d(L, v, dtype, pad_weights_2d(w, ry, rx, R), R, R, edge, pad, in, out, rows, cols);
  }
  switch (ry) {
    case 1: return launch_overlap2d_tiled<1>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 2: return launch_overlap2d_tiled<2>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 3: return launch_overlap2d_tiled<3>(L, v, dtype, w, edge, pad, in, out, rows, cols);
    case 4: return launch_overlap2d_tiled<4>(L, v, dtype, w, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

}  // namespace skel
