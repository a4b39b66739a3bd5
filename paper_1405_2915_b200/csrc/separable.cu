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
#include <string.h>

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
                       int rows, int cols, int tiles_x, int ntiles, unsigned* tile_ctr, unsigned tile_base,
                       int frame_tiles_y /* 0: all tiles; > 2: only the tiles on the border of a tiles_x x frame_tiles_y grid */) {
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
      int y = int(t) / tiles_x, x = int(t) - y * tiles_x;
      if (frame_tiles_y) {  // t counts the border tiles: first row, last row, then (left, right) of every row between
        if (y == 1) y = frame_tiles_y - 1;
        else if (y >= 2) {
          const int g = int(t) - 2 * tiles_x;
          y = 1 + g / 2;
          x = (g & 1) ? tiles_x - 1 : 0;
        }
      }
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
                       float* out, size_t rows, size_t cols, bool frame_only = false) {
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
  const size_t tiles_x = (cols + T2_TW - 1) / T2_TW, tiles_y = (rows + S::TH - 1) / S::TH;
  const bool frame = frame_only && tiles_x > 2 && tiles_y > 2;   // small matrices: every tile touches the border anyway
  const size_t ntiles = frame ? 2 * tiles_x + 2 * (tiles_y - 2) : tiles_x * tiles_y;
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T2_THREADS, S::SMEM, L.stream>>>(wrow, wcol, tmap, edge, pad, in, out, (int)rows, (int)cols,
                                                          (int)tiles_x, (int)ntiles, L.tile_ctr, *L.tile_next,
                                                          frame ? (int)tiles_y : 0);
  *L.tile_next += unsigned(ntiles);  // ntiles - grid ids fetched from the counter + one failing fetch per block
  ++*L.launches;
  return cudaGetLastError();
}

// ---- register-marching form ("march_r8") ----------------------------------------------------------------------------
// One WARP per 128-column strip walks down a segment of L output rows; nothing of the intermediate T ever touches shared
// memory. Per window row the warp reads its 4 + 16 window columns from its own ring of bulk tensor copies (3 stages of
// 8 rows x 144 columns per warp, TMA; the warp that consumes a stage re-arms it, so there is no `empty` barrier and no
// block barrier at all), computes the row pass of 4 columns per lane (broadcast FFMA2, two chains), and feeds the 4
// values into the 17 column-pass accumulators of the 17 output rows that are in flight (68 registers; the row that
// receives its last tap is stored). The accumulator a T row goes to depends on (row mod 17), so the row loop is unrolled
// 17 times and the rotation costs no moves. Every output receives the same taps in the same order as the two 1D calls
// (row pass ascending from zero, rounded to fp32, column pass ascending from zero): bit-identical to them. The row pass
// is recomputed for the 16 halo rows of a segment only (L = 222 at 8192^2: 7 %), against 25 - 50 % for the tiled forms.
// Borders: the marching kernel sees zeros outside the matrix (the tensor copy's fill) and T = 0 in rows outside it,
// which IS the CONSTANT policy with pad = 0. CONSTANT with another pad and DUPLICATE are applied in registers when the
// columns fill whole strips (kernel MODE 1 / 2 below). For CYCLIC and for ragged column counts the outputs within MR
// rows / columns of the border (the only ones that see cells outside the matrix) come out wrong, and a second launch
// recomputes the 32 x 128 tiles on the border of the matrix with the tiled fused kernel above, which patches its windows
// with the edge policy (4 % of the tiles at 8192^2). Patching the stages inside the marching loop would need calls, and
// a call with 100 live registers spills them.
constexpr int MR = 8, MFW = 2 * MR + 1, M_KROWS = 8, M_NS = 3, M_SWC = 128 + 2 * MR;   // 144 floats per staged row
constexpr unsigned M_STAGE_BYTES = M_KROWS * M_SWC * 4;                                  // 4608
struct WPairs1D { float2 p[MFW + 1]; };  // p[d] = (w[d], w[d-1]) with w[-1] = w[17] = 0

__device__ __forceinline__ void mbar_wait_s(uint32_t bar, unsigned parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_LOOP:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra WAIT_DONE;\nbra WAIT_LOOP;\nWAIT_DONE:\n}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void march_refill(uint32_t dst, uint32_t bar, const CUtensorMap* map, int x, int y) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(M_STAGE_BYTES) : "memory");
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
               "l"(map), "r"(x), "r"(y), "r"(bar)
               : "memory");
}
__device__ __forceinline__ float lds32_s(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts64_s(uint32_t addr, float a, float b) {
  asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ float4 lds128_s(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
// MODE 0: cells outside the matrix are zeros (what the tensor copy delivers) and T is 0 in rows outside it: CONSTANT 0.
// MODE 1 (CONSTANT, pad != 0) and MODE 2 (DUPLICATE), cols % 128 == 0: the policy is applied in REGISTERS. Columns: only
// lanes 0, 1 of the first strip and lanes 30, 31 of the last strip hold window columns outside the matrix, and the
// element that DUPLICATE repeats (column 0 / cols - 1) is in the lane's own window. Rows: a T row outside the matrix
// is `pad` (MODE 1) or the T of row 0 / rows - 1 (MODE 2: the last row's T is simply kept; the first row's T is computed
// before the walk starts, from the second chunk of the ring).
__device__ __forceinline__ void march_rowpass(const WPairs1D& Wr, const float (&v)[20], float (&t)[4]) {
  constexpr int FW = MFW;
  t[0] = t[1] = t[2] = t[3] = 0.f;
#pragma unroll
  for (int d = 0; d <= FW; ++d) {   // broadcast form: outputs (2j, 2j+1) take window element v[d + 2j] with taps d and d - 1
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const float x = v[d + 2 * j];
      if (d == 0) t[2 * j] = fmaf(Wr.p[0].x, x, t[2 * j]);
      else if (d == FW) t[2 * j + 1] = fmaf(Wr.p[FW].y, x, t[2 * j + 1]);
      else fma2_bcast(t[2 * j], t[2 * j + 1], Wr.p[d], x);
    }
  }
}
template <int MODE>
__device__ __forceinline__ void march_fix_cols(float (&v)[20], int lane, bool left, bool right, float pad) {
  if (left && lane < 2) {          // lane 0: window columns -8 .. 11, lane 1: -4 .. 15
    const float x0 = MODE == 1 ? pad : (lane == 0 ? v[8] : v[4]);
#pragma unroll
    for (int j = 0; j < 8; ++j)
      if (j < 4 || lane == 0) v[j] = x0;
  }
  if (right && lane >= 30) {       // lane 30: columns cols - 16 .. cols + 3, lane 31: cols - 12 .. cols + 7
    const float x1 = MODE == 1 ? pad : (lane == 31 ? v[11] : v[15]);
#pragma unroll
    for (int j = 12; j < 20; ++j)
      if (j >= 16 || lane == 31) v[j] = x1;
  }
}

// Columns outside the matrix (MODE 1 / 2): the first and the last strip of a row of strips patch the 8 outside columns of
// each chunk in their stage when it lands (64 cells, two per lane), then fence.proxy.async before the stage is re-armed.
// (The same fix-up on the window registers of every row, as predicated selects, cost 12 % of the kernel; a separate copy
// of the row loop for the border strips made them the stragglers: two 46 KB instruction streams on their SMs.)
template <int MODE>
__device__ __forceinline__ void march_strip(const WPairs1D& Wr, const Weights1D& Wc, const CUtensorMap* tmap, float* out, int rows,
                                            int cols, int L, int nstrips, float pad, unsigned char* ring, uint64_t* full,
                                            int seg, int strip) {
  constexpr int R = MR, FW = MFW, KROWS = M_KROWS, NS = M_NS, SWC = M_SWC;
  constexpr unsigned STAGE_BYTES = M_STAGE_BYTES;
  const int lane = threadIdx.x & 31;
  const int r0 = seg * L, c0 = strip * 128;
  const int nout = min(L, rows - r0);
  const int nwin = nout + 2 * R;                  // window rows r0 - R .. r0 + nout + R - 1
  const int nchunks = (nwin + KROWS - 1) / KROWS;
  const uint32_t ring32 = smem_u32(ring), sbase = ring32 + lane * 16, full32 = smem_u32(full);
  if (lane == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(full + s, 1);
    mbar_fence_init();
    for (int s = 0; s < NS && s < nchunks; ++s) march_refill(ring32 + s * STAGE_BYTES, full32 + 8 * s, tmap, c0 - R, r0 - R + s * KROWS);
  }
  __syncwarp();
  const bool col_ok = c0 + lane * 4 < cols;       // cols % 4 == 0: a lane's 4 columns are inside or outside together
  float acc[FW][4];
#pragma unroll
  for (int s = 0; s < FW; ++s)
#pragma unroll
    for (int e = 0; e < 4; ++e) acc[s][e] = 0.f;
  float* optr = out + (static_cast<long long>(r0) - 2 * R) * cols + c0 + lane * 4;  // output row of window row `row`, minus 2R
  uint32_t off = 0, st_off = 0;   // byte offsets in the ring of the current row and of the current stage
  int rin = 0, chunk = 0;
  uint32_t bar = full32;
  unsigned ph = 0;
  int prow = r0 - R;
  const bool left = strip == 0, right = strip == nstrips - 1;
  float tk[4] = {0.f, 0.f, 0.f, 0.f};   // MODE 2: the T a row outside the matrix takes (row 0's before the matrix, the last row's after)
  if (MODE == 2 && r0 == 0) {           // matrix row 0 is window row R = row 0 of the second chunk (R == KROWS)
    mbar_wait_s(full32 + 8, 0);
    float v[20];
#pragma unroll
    for (int g = 0; g < 5; ++g) {
      const float4 t4 = lds128_s(sbase + STAGE_BYTES + 16 * g);
      v[4 * g] = t4.x; v[4 * g + 1] = t4.y; v[4 * g + 2] = t4.z; v[4 * g + 3] = t4.w;
    }
    march_fix_cols<MODE>(v, lane, left, right, pad);   // (chunk 1 is patched in shared memory only when the walk reaches it)
    march_rowpass(Wr, v, tk);
  }
  for (int q = 0; q < nwin; q += FW) {
#pragma unroll
    for (int k = 0; k < FW; ++k) {
      const int row = q + k;
      if (row < nwin) {
        if (rin == 0) {
          mbar_wait_s(bar, ph);
          if (MODE != 0 && (left || right)) {   // warp-uniform, once per chunk
            const uint32_t a = ring32 + st_off + (lane >> 2) * (SWC * 4) + (lane & 3) * 8;   // row lane / 4, cells 2 (lane % 4), + 1
            if (left) {
              const float x0 = MODE == 1 ? pad : lds32_s(ring32 + st_off + (lane >> 2) * (SWC * 4) + R * 4);
              sts64_s(a, x0, x0);
            }
            if (right) {
              const float x1 = MODE == 1 ? pad : lds32_s(ring32 + st_off + (lane >> 2) * (SWC * 4) + (R + 127) * 4);
              sts64_s(a + (R + 128) * 4, x1, x1);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes before the stage is re-armed
            __syncwarp();
          }
        }
        float v[20];
#pragma unroll
        for (int g = 0; g < 5; ++g) {
          const float4 t4 = lds128_s(sbase + off + 16 * g);
          v[4 * g] = t4.x; v[4 * g + 1] = t4.y; v[4 * g + 2] = t4.z; v[4 * g + 3] = t4.w;
        }
        if (rin == KROWS - 1) {  // the warp is done with this stage: re-arm it with chunk + NS
          __syncwarp();
          if (lane == 0 && chunk + NS < nchunks) march_refill(ring32 + st_off, bar, tmap, c0 - R, r0 - R + (chunk + NS) * KROWS);
          rin = 0; ++chunk; st_off += STAGE_BYTES; bar += 8;
          if (st_off == NS * STAGE_BYTES) { st_off = 0; bar = full32; ph ^= 1u; }
        } else {
          ++rin;
        }
        off += SWC * 4;
        if (off == NS * KROWS * SWC * 4) off = 0;
        float t[4];
        march_rowpass(Wr, v, t);
        if (prow < 0 || prow >= rows) {   // a T row outside the matrix
#pragma unroll
          for (int e = 0; e < 4; ++e) t[e] = MODE == 0 ? 0.f : (MODE == 1 ? pad : tk[e]);
        } else if (MODE == 2) {
#pragma unroll
          for (int e = 0; e < 4; ++e) tk[e] = t[e];   // rows after the matrix repeat the last row's T
        }
        ++prow;
        // column pass: T row `row` is tap a of output m = row - a, accumulator (k - a) mod 17
#pragma unroll
        for (int a = 0; a < FW; ++a) {
          const int slot = (k - a + FW) % FW;
          if (a == 0) acc[slot][0] = acc[slot][1] = acc[slot][2] = acc[slot][3] = 0.f;
          fma2_into(acc[slot][0], acc[slot][1], Wc.w[a], t[0], t[1]);
          fma2_into(acc[slot][2], acc[slot][3], Wc.w[a], t[2], t[3]);
        }
        if (row >= 2 * R && col_ok) {
          const int slot = (k - 2 * R + FW) % FW;
          uint32_t raw[4] = {__float_as_uint(acc[slot][0]), __float_as_uint(acc[slot][1]), __float_as_uint(acc[slot][2]),
                             __float_as_uint(acc[slot][3])};
          st_stream<4>(optr, raw);
        }
        optr += cols;
      }
    }
  }
}

template <int MODE>
__global__ void __launch_bounds__(256, 2)
separable_march_kernel(const __grid_constant__ WPairs1D Wr, const __grid_constant__ Weights1D Wc,
                       const __grid_constant__ CUtensorMap tmap, float* out, int rows, int cols, int L, int nstrips,
                       int ntasks, float pad) {
  extern __shared__ __align__(128) unsigned char smraw[];
  const int warp = threadIdx.x >> 5;
  unsigned char* ring = smraw + warp * (M_NS * M_STAGE_BYTES);
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw + 8 * M_NS * M_STAGE_BYTES) + warp * M_NS;
  const int task = blockIdx.x * 8 + warp;
  if (task >= ntasks) return;   // no block-wide barrier anywhere below
  const int seg = task / nstrips, strip = task - seg * nstrips;
  march_strip<MODE>(Wr, Wc, &tmap, out, rows, cols, L, nstrips, pad, ring, full, seg, strip);
}

cudaError_t launch_sep_march(const Launch& L, const Weights1D& wrow, const Weights1D& wcol, int edge, float pad, const float* in,
                             float* out, size_t rows, size_t cols) {
  constexpr size_t smem = 8 * M_NS * M_STAGE_BYTES + 8 * M_NS * sizeof(uint64_t);
  uint32_t pad_bits;
  memcpy(&pad_bits, &pad, 4);
  const bool zeros_outside = edge == EDGE_CONSTANT && pad_bits == 0u;   // +0.0 only: the fill of the tensor copy
  // the second launch redoes the border TILES: they cover the frame only if the last (ragged) tile row / column holds
  // at least MR rows / columns; other shapes, and matrices of at most two tiles in a direction, run the tiled kernel alone
  const bool frame_in_border_tiles = (rows % 32 == 0 || rows % 32 >= MR) && (cols % T2_TW == 0 || cols % T2_TW >= MR) &&
                                     (cols + T2_TW - 1) / T2_TW > 2 && (rows + 31) / 32 > 2;
  // in-register policy (kernel MODE 1 / 2): CONSTANT and DUPLICATE on matrices whose columns fill whole strips
  const int mode = zeros_outside ? 0 : (cols % 128 == 0 && edge == EDGE_CONSTANT ? 1 : (cols % 128 == 0 && edge == EDGE_DUPLICATE ? 2 : 0));
  if (!zeros_outside && mode == 0 && !frame_in_border_tiles) return launch_sep<MR, 4, 1>(L, wrow, wcol, edge, pad, in, out, rows, cols);
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(separable_march_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(separable_march_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(separable_march_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, separable_march_kernel<2>, 256, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tmap;
  cudaError_t e = make_tmap_2d(&tmap, in, rows, cols, M_SWC, M_KROWS);
  if (e != cudaSuccess) return e;
  WPairs1D P;
  for (int d = 0; d <= MFW; ++d) {
    P.p[d].x = d < MFW ? wrow.w[d] : 0.f;
    P.p[d].y = d >= 1 ? wrow.w[d - 1] : 0.f;
  }
  // segments: whole waves of (SMs x resident blocks x 8) warps when the matrix is large enough, segments of about 224
  // rows (7 % halo), never shorter than 32 rows
  const size_t nstrips = (cols + 127) / 128;
  const size_t slots = size_t(L.sms) * per_sm * 8;
  const size_t per_wave = slots / nstrips > 0 ? slots / nstrips : 1;
  const size_t want = (rows + 223) / 224;
  const size_t waves = (want + per_wave - 1) / per_wave;
  size_t nseg = waves * per_wave;
  const size_t max_seg = (rows + 31) / 32;
  if (nseg > max_seg) nseg = max_seg;
  const size_t Lrows = (rows + nseg - 1) / nseg;
  nseg = (rows + Lrows - 1) / Lrows;
  const size_t ntasks = nstrips * nseg;
  const size_t grid = (ntasks + 7) / 8;
  if (mode == 1)
    separable_march_kernel<1><<<(unsigned)grid, 256, smem, L.stream>>>(P, wcol, tmap, out, (int)rows, (int)cols, (int)Lrows,
                                                                        (int)nstrips, (int)ntasks, pad);
  else if (mode == 2)
    separable_march_kernel<2><<<(unsigned)grid, 256, smem, L.stream>>>(P, wcol, tmap, out, (int)rows, (int)cols, (int)Lrows,
                                                                        (int)nstrips, (int)ntasks, pad);
  else
    separable_march_kernel<0><<<(unsigned)grid, 256, smem, L.stream>>>(P, wcol, tmap, out, (int)rows, (int)cols, (int)Lrows,
                                                                        (int)nstrips, (int)ntasks, pad);
  ++*L.launches;
  if (!zeros_outside && mode == 0)  // the border tiles again, with the edge policy (they are a superset of the frame)
    return launch_sep<MR, 4, 1>(L, wrow, wcol, edge, pad, in, out, rows, cols, true);
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

const char* const kSepNames[] = {"two_pass", "fused_oy4", "fused_oy8", "fused_oy4_s1", "fused_oy8_s1", "march_r8"};
constexpr int kNumSep = 6;

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
  if (v == 5)  // the marching form exists for radius 8; smaller radii run it zero-padded (kernels.hpp)
    return launch_sep_march(L, pad_weights_1d(wrow, r_row, MR), pad_weights_1d(wcol, r_col, MR), edge, pad, in, out, rows, cols);
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
