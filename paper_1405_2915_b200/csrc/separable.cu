// Fused separable MapOverlap on a matrix (BASELINE.json configs[3] "separable
// row-then-column 1D passes"): out = colpass(w_col, RN_f32(rowpass(w_row, X))) with the edge policy
// applied by each pass, i.e. exactly what skel_mapoverlap_1d_matrix(ROW) into a temporary followed
// by skel_mapoverlap_1d_matrix(COL) computes, but the fp32 intermediate T lives in shared memory:
// 8 B/elem of HBM traffic instead of 16.
//
// Persistent blocks walk 8*OY x 128 output tiles. Per tile: ONE 2-D tensor copy (TMA) brings the
// (8*OY + 2r) x (128 + 2*ceil4(r)) window of X into one of two stages (out-of-range cells arrive as
// zeros and are patched with the edge policy on border tiles); phase A computes the row pass of
// every window row into T (8*OY + 2r rows x 128, shared memory), phase B the column pass from T to
// global memory (the column kernel's register-blocked form: 4 x OY outputs per thread). Rows of T
// outside the matrix are, per policy: CONSTANT -> pad (not rowpass(pad)); DUPLICATE / CYCLIC -> the
// row pass of the clamped / wrapped row, which is what the patched window holds.
// Taps accumulate in ascending order from zero in both passes, like the 1D kernels.
#include "overlap2d_tiles.cuh"

namespace skel {
namespace {

template <int R, int OY, int STAGES> struct SepGeom {
  using G = Tile2Geom<R, R, OY>;
  static constexpr int RXP = G::RXP, TH = G::TH, SW = G::SW, SH = G::SH;
  static constexpr unsigned T_BYTES = unsigned(SH) * T2_TW * 4u;
  static constexpr size_t SMEM = STAGES * size_t(G::STAGE_STRIDE) + T_BYTES + 6 * sizeof(uint64_t);  // + full/empty, coord
};

// STAGES = 2: the window of tile i+1 is requested while tile i is in phase A (full/empty mbarriers).
// STAGES = 1: one window buffer; the next window is requested as soon as phase A has consumed the
// current one and lands during phase B. Half the shared memory, so twice the resident blocks.
template <int R, int OY, int STAGES>
__global__ void __launch_bounds__(T2_THREADS)
separable_fused_kernel(const __grid_constant__ Weights1D Wrow, const __grid_constant__ Weights1D Wcol,
                       const __grid_constant__ CUtensorMap tmap, int edge, float pad, const float* in, float* out,
                       int rows, int cols, int tiles_x, int ntiles, unsigned* tile_ctr, unsigned tile_base) {
  using S = SepGeom<R, OY, STAGES>;
  using G = typename S::G;
  constexpr int RXP = S::RXP, TH = S::TH, SW = S::SW, SH = S::SH;
  constexpr int NGX = (4 + 2 * RXP) / 4;
  extern __shared__ __align__(128) unsigned char smraw[];
  float* T = reinterpret_cast<float*>(smraw + STAGES * G::STAGE_STRIDE);
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw + STAGES * G::STAGE_STRIDE + S::T_BYTES);
  uint64_t* empty = full + 2;
  int2* coord = reinterpret_cast<int2*>(empty + 2);  // (r0, c0) of the tile in each stage; r0 < 0: no more tiles
  auto stage_ptr = [&](int s) { return reinterpret_cast<float*>(smraw + s * G::STAGE_STRIDE); };
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    for (int s = 0; s < 2; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, T2_THREADS / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();
  // dynamic tile assignment (see overlap2d_tma_kernel): first tile = block index, then a global counter, fetched one
  // tile ahead of its use; exactly one failing fetch per block
  unsigned t_next = blockIdx.x;
  bool exhausted = false;
  auto produce = [&](int s) {  // thread 0
    const unsigned t = t_next;
    if (!exhausted) exhausted = t >= unsigned(ntiles);
    if (!exhausted) t_next = atomicAdd(tile_ctr, 1u) - tile_base + gridDim.x;
    if (!exhausted) {
      const int y = int(t) / tiles_x, x = int(t) - y * tiles_x;
      coord[s] = make_int2(y * TH, x * T2_TW);
      mbar_arrive_expect_tx(full + s, G::STAGE_BYTES);
      tma_load_2d(stage_ptr(s), &tmap, x * T2_TW - RXP, y * TH - R, full + s);
    } else {
      coord[s] = make_int2(-1, 0);
      mbar_arrive(full + s);
    }
  };
  if (threadIdx.x == 0) produce(0);
  const bool patch_needed = !(edge == EDGE_CONSTANT && bits_are_zero(pad));
  int s = 0, ph = 0, tph = 1;
  for (int it = 0;; ++it) {
    if (STAGES == 2 && threadIdx.x == 0) {
      if (it > 0) mbar_wait(empty + (s ^ 1), tph);
      produce(s ^ 1);
    }
    if (s == 0) tph ^= 1;  // parity of the next wait on an `empty` barrier (see overlap2d_tma_kernel)
    mbar_wait(full + s, ph);
    const int2 rc = coord[s];
    if (rc.x < 0) break;
    const int r0 = rc.x, c0 = rc.y;
    float* sm = stage_ptr(s);
    const bool window_inside = r0 - R >= 0 && r0 + TH + R <= rows && c0 - RXP >= 0 && c0 + T2_TW + RXP <= cols;
    if (!window_inside && patch_needed) {
      for (int idx = threadIdx.x; idx < SH * SW; idx += T2_THREADS) {
        const int gy = idx / SW, gx = idx - gy * SW;
        const int p = r0 - R + gy, q = c0 - RXP + gx;
        if (p < 0 || p >= rows || q < 0 || q >= cols) sm[idx] = ext2(in, rows, cols, p, q, edge, pad);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();
    }
    // ---- phase A: row pass of window row gy into T (warp w takes rows w, w+8, ...) ----
    for (int gy = warp; gy < SH; gy += T2_THREADS / 32) {
      const float* srow = sm + gy * SW + lane * 4;
      float v[4 * NGX];
#pragma unroll
      for (int g = 0; g < NGX; ++g) {
        const float4 t = *reinterpret_cast<const float4*>(srow + 4 * g);
        v[4 * g] = t.x; v[4 * g + 1] = t.y; v[4 * g + 2] = t.z; v[4 * g + 3] = t.w;
      }
      float p[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int b = 0; b <= 2 * R; ++b) {
        if ((RXP - R + b) % 2 == 0) {
          fma2_into(p[0], p[1], Wrow.w[b], v[RXP - R + b], v[RXP - R + b + 1]);
          fma2_into(p[2], p[3], Wrow.w[b], v[RXP - R + b + 2], v[RXP - R + b + 3]);
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) p[e] = fmaf(Wrow.w[b], v[RXP - R + b + e], p[e]);
        }
      }
      const int prow = r0 - R + gy;
      if (edge == EDGE_CONSTANT && (prow < 0 || prow >= rows)) p[0] = p[1] = p[2] = p[3] = pad;
      *reinterpret_cast<float4*>(T + gy * T2_TW + lane * 4) = make_float4(p[0], p[1], p[2], p[3]);
    }
    if constexpr (STAGES == 2) {
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + s);  // this warp no longer reads the X stage
    }
    __syncthreads();  // T is complete (and, with one stage, nobody reads the window any more)
    if (STAGES == 1 && threadIdx.x == 0) produce(0);  // everybody has read coord[0] and the window
    // ---- phase B: column pass from T (a (2R+1) x 1 filter on a tile without x halo) ----
    compute_tile2<R, 0, OY, Weights1D, true>(T, Wcol, out, rows, cols, r0, c0, r0 + TH <= rows && c0 + T2_TW <= cols);
    __syncthreads();  // T is rewritten by the next tile's phase A
    if constexpr (STAGES == 2) {
      s ^= 1;
      if (s == 0) ph ^= 1;
    } else {
      ph ^= 1;
    }
  }
}

template <int R, int OY, int STAGES>
cudaError_t launch_sep(const Launch& L, const Weights1D& wrow, const Weights1D& wcol, int edge, float pad, const float* in,
                       float* out, size_t rows, size_t cols) {
  using S = SepGeom<R, OY, STAGES>;
  static_assert(S::SMEM <= 227 * 1024, "does not fit");
  auto kern = separable_fused_kernel<R, OY, STAGES>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T2_THREADS, S::SMEM) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tmap;
  cudaError_t e = make_tmap_2d(&tmap, in, rows, cols, S::SW, S::SH);
  if (e != cudaSuccess) return e;
  const size_t tiles_x = (cols + T2_TW - 1) / T2_TW;
  const size_t ntiles = tiles_x * ((rows + S::TH - 1) / S::TH);
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T2_THREADS, S::SMEM, L.stream>>>(wrow, wcol, tmap, edge, pad, in, out, (int)rows, (int)cols,
                                                          (int)tiles_x, (int)ntiles, L.tile_ctr, *L.tile_next);
  *L.tile_next += unsigned(ntiles);  // ntiles - grid ids fetched from the counter + one failing fetch per block
  ++*L.launches;
  return cudaGetLastError();
}

template <int R>
cudaError_t launch_sep_r(const Launch& L, int v, const Weights1D& wrow, const Weights1D& wcol, int edge, float pad,
                         const float* in, float* out, size_t rows, size_t cols) {
  if (v == 1) return launch_sep<R, 4, 2>(L, wrow, wcol, edge, pad, in, out, rows, cols);
  if (v == 2) return launch_sep<R, 8, 2>(L, wrow, wcol, edge, pad, in, out, rows, cols);
  if (v == 3) return launch_sep<R, 4, 1>(L, wrow, wcol, edge, pad, in, out, rows, cols);
  if (v == 4) return launch_sep<R, 8, 1>(L, wrow, wcol, edge, pad, in, out, rows, cols);
  return cudaErrorInvalidValue;
}

const char* const kSepNames[] = {"two_pass", "fused_oy4", "fused_oy8", "fused_oy4_s1", "fused_oy8_s1"};
constexpr int kNumSep = 5;

}  // namespace

int separable_variant_count() { return kNumSep; }
const char* separable_variant_name(int v) { return (v >= 0 && v < kNumSep) ? kSepNames[v] : nullptr; }
bool separable_variant_ok(int v, int r_row, int r_col, const void* in, const void* out, size_t rows, size_t cols) {
  if (v < 0 || v >= kNumSep) return false;
  if (v == 0) return true;
  // unequal radii and radii between the instantiated ones run zero-padded to the next of {1, 2, 3, 4, 8} (kernels.hpp)
  const bool templated = r_row >= 0 && r_col >= 0 && r_row <= 8 && r_col <= 8;
  return templated && reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0 &&
         cols % 4 == 0 && rows < (size_t(1) << 30) && cols < (size_t(1) << 30) &&
         ((rows + 31) / 32) * ((cols + 127) / 128) < (size_t(1) << 30);
}

cudaError_t launch_separable_fused(const Launch& L, int v, const Weights1D& wrow, const Weights1D& wcol, int r_row,
                                   int r_col, int edge, float pad, const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  const int rmax = r_row > r_col ? r_row : r_col;
  const int r = rmax <= 4 ? (rmax < 1 ? 1 : rmax) : (rmax <= 8 ? 8 : -1);
  if (r != r_row || r != r_col)  // zero-padded to the next instantiated radius (kernels.hpp)
    return launch_separable_fused(L, v, pad_weights_1d(wrow, r_row, r), pad_weights_1d(wcol, r_col, r), r, r, edge, pad, in,
                                  out, rows, cols);
  switch (r) {
    case 1: return launch_sep_r<1>(L, v, wrow, wcol, edge, pad, in, out, rows, cols);
    case 2: return launch_sep_r<2>(L, v, wrow, wcol, edge, pad, in, out, rows, cols);
    case 3: return launch_sep_r<3>(L, v, wrow, wcol, edge, pad, in, out, rows, cols);
    case 4: return launch_sep_r<4>(L, v, wrow, wcol, edge, pad, in, out, rows, cols);
    case 8: return launch_sep_r<8>(L, v, wrow, wcol, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

}  // namespace skel
