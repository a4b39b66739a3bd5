// MapOverlap 1D skeleton on a vector or along the rows of a matrix (PAPER.md L83 names
// "mapoverlap"; definition: DESIGN.md reading 5):
//   out[i] = sum_{k=-r..r} w[k+r] * x~[i+k]      (correlation; edge policy constant(pad) | duplicate | cyclic)
// Every row of a rows x cols matrix is an independent vector (a plain vector is rows = 1).
//
// Variants:
//  * "direct": any r <= 64, any alignment. One output per thread, coalesced; the 2r+1 neighbour
//    loads of a warp overlap and are served by L1.
//  * "tiled_o{4,8,16}": the tile plus a halo is staged once in shared memory with 128-bit loads;
//    every thread then produces O consecutive outputs from a register window that slides over
//    128-bit shared-memory reads ((O + 2*ceil4(r))/4 reads per O outputs), weights come from the
//    constant bank, taps are fully unrolled (r is a template parameter: 1,2,3,4,8,16).
//    The tile is padded by 4 floats every O floats so that the 128-bit reads of a quarter warp
//    fall into distinct banks.
#include <cuda.h>
#include "common.cuh"
#include "kernels.hpp"

namespace skel {
namespace {

enum : int { EDGE_CONSTANT = 0, EDGE_DUPLICATE = 1, EDGE_CYCLIC = 2 };

// x~ of one row (reading 5): c may be out of [0, cols)
__device__ __forceinline__ float ext_row(const float* row, long long cols, long long c, int edge, float pad) {
  if (c >= 0 && c < cols) return __ldg(row + c);
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) {  // non-negative remainder: the index wraps around (possibly several times)
    long long m = c % cols;
    return __ldg(row + (m < 0 ? m + cols : m));
  }
  return __ldg(row + (c < 0 ? 0 : cols - 1));
}

// ---- direct --------------------------------------------------------------------------------
// Up to 33 taps (r <= 16) are ONE chain in ascending tap order, like every tiled variant (so all variants, and the
// fused separable kernel, give the same bits; bound 33 * 2^-24 = 1.97e-6 of sum|w x|). Longer filters are chained in
// groups of 16 taps and the group sums added: (16 + #groups - 1) * 2^-24 <= 1.44e-6.
template <typename T>
__global__ void __launch_bounds__(256)
overlap1d_direct_kernel(const __grid_constant__ Weights1D W, int r, int edge, float pad, const float* in, float* out,
                        size_t rows, size_t cols) {
  const size_t total = rows * cols;
  for (size_t idx = blockIdx.x * size_t(blockDim.x) + threadIdx.x; idx < total; idx += size_t(gridDim.x) * blockDim.x) {
    const size_t row = idx / cols;
    const long long j = static_cast<long long>(idx - row * cols);
    const float* x = in + row * cols;
    float total_acc = 0.f;
    const bool interior = (j - r >= 0) && (j + r < static_cast<long long>(cols));
    const int chain = 2 * r + 1 <= 33 ? 33 : 16;
    for (int k0 = 0; k0 <= 2 * r; k0 += chain) {
      const int k1 = min(k0 + chain, 2 * r + 1);
      float acc = 0.f;
      if (interior) {
        for (int k = k0; k < k1; ++k) acc = StencilOps<T>::mad(W.w[k], __ldg(x + j + k - r), acc);
      } else {
        for (int k = k0; k < k1; ++k) acc = StencilOps<T>::mad(W.w[k], ext_row(x, (long long)cols, j + k - r, edge, pad), acc);
      }
      total_acc = k0 == 0 ? acc : StencilOps<T>::add(total_acc, acc);
    }
    out[idx] = total_acc;
  }
}

// ---- shared-memory tiled ---------------------------------------------------------------------
constexpr int T1_THREADS = 256;

template <int O> __device__ __forceinline__ int phys(int sc) {  // padded smem index of tile coordinate sc
  if constexpr (O == 4) return sc;
  else return sc + 4 * (sc / O);
}

// stage x~[c0 - HP, c0 + TILE + HP) of one row at tile coordinates sc = 0 .. SPAN-1 (padded layout).
// ASYNC: in-range 128-bit groups go through cp.async (LDGSTS), edge groups are computed and stored.
template <int R, int O, bool ASYNC>
__device__ __forceinline__ void stage_tile1(float* sm, const float* x, long long cols, long long c0, int edge, float pad) {
  constexpr int HP = (R + 3) / 4 * 4;
  constexpr int SPAN = T1_THREADS * O + 2 * HP;
  for (int g = threadIdx.x; g < SPAN / 4; g += T1_THREADS) {
    const long long c = c0 - HP + 4 * g;
    float* dst = sm + phys<O>(4 * g);
    if (c >= 0 && c + 3 < cols) {
      if constexpr (ASYNC) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(x + c) : "memory");
      } else {
        uint32_t raw[4];
        ld_stream<4, true>(raw, x + c);
        *reinterpret_cast<float4*>(dst) =
            make_float4(__uint_as_float(raw[0]), __uint_as_float(raw[1]), __uint_as_float(raw[2]), __uint_as_float(raw[3]));
      }
    } else {
      float4 v;
      v.x = ext_row(x, cols, c, edge, pad);
      v.y = ext_row(x, cols, c + 1, edge, pad);
      v.z = ext_row(x, cols, c + 2, edge, pad);
      v.w = ext_row(x, cols, c + 3, edge, pad);
      *reinterpret_cast<float4*>(dst) = v;
    }
  }
}

// thread t produces outputs c0 + t*O .. + O-1 from tile coordinates t*O .. t*O + O + 2HP - 1
// packed fp32 pair (Blackwell FFMA2): (lo, hi) += w * (x0, x1), one instruction on an aligned register pair
__device__ __forceinline__ void fma2_into(float& lo, float& hi, float w, float x0, float x1) {
  unsigned long long ww, xx, cc, d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ww) : "f"(w), "f"(w));
  asm("mov.b64 %0, {%1, %2};" : "=l"(xx) : "f"(x0), "f"(x1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(cc) : "f"(lo), "f"(hi));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(ww), "l"(xx), "l"(cc));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}

// thread t produces outputs c0 + t*O .. + O-1 from tile coordinates t*O .. t*O + O + 2HP - 1.
// PK: the FMAs (x[p] -> out o) and (x[p+1] -> out o+1) with p, o even share the tap and are ONE FFMA2
// on two aligned register pairs; the other half of the FMAs stays scalar. Emission order keeps, for
// every output, its taps in ascending order, so the result is bit-identical to the scalar form.
// SWZ >= 0: the tile is a TMA window of 128-byte rows in the 128-byte swizzle (16-byte chunk c of row q sits at
// chunk c ^ (q & 7)); the thread's first group is chunk threadIdx.x * O / 4 + SWZ of the window. With u = t + a
// (a = (SWZ + g) / 4, b = (SWZ + g) % 4; O = 16) the group's byte address is ((u >> 1) * 128 | (((u & 1) * 4) ^
// ((u >> 1) & 7)) * 16) ^ (b * 16): one XOR per group on top of five integer instructions per a.
template <int R, int O, bool PK_ = false, int SWZ = -1, typename T = float>
__device__ __forceinline__ void compute_tile1(const float* sm, const Weights1D& W, float* orow, long long cols, long long c0) {
  constexpr int HP = (R + 3) / 4 * 4;
  constexpr int NG = (O + 2 * HP) / 4;  // 128-bit groups a thread reads
  constexpr bool PK = PK_ && StencilOps<T>::kFloat;
  static_assert(SWZ < 0 || O == 16, "the swizzled window form is written for 16 outputs per thread");
  float acc[O];
#pragma unroll
  for (int o = 0; o < O; ++o) acc[o] = 0.f;
  const int sc0 = threadIdx.x * O;
  unsigned swz_a[SWZ >= 0 ? (SWZ + NG + 3) / 4 : 1];
  if constexpr (SWZ >= 0) {
#pragma unroll
    for (int a = 0; a < (SWZ + NG + 3) / 4; ++a) {
      const unsigned u = threadIdx.x + a, q = u >> 1;
      swz_a[a] = (q << 7) | ((((u & 1u) << 2) ^ (q & 7u)) << 4);
    }
  }
#pragma unroll
  for (int g = 0; g < NG; ++g) {
    float4 v4;
    if constexpr (SWZ >= 0)
      v4 = *reinterpret_cast<const float4*>(reinterpret_cast<const unsigned char*>(sm) +
                                            (swz_a[(SWZ + g) / 4] ^ (unsigned((SWZ + g) % 4) << 4)));
    else
      v4 = *reinterpret_cast<const float4*>(sm + phys<O>(sc0 + 4 * g));
    const float v[4] = {v4.x, v4.y, v4.z, v4.w};
    // tile coordinate (relative to sc0) p = 4g+e holds x~[out0 - HP + p]; output o uses it with
    // tap k = p - HP - o + R, 0 <= k <= 2R
    if constexpr (PK) {
#pragma unroll
      for (int e = 0; e < 4; e += 2) {
#pragma unroll
        for (int o = 1; o < O; o += 2) {  // x[p] -> odd outputs (scalar), before their paired tap p+1
          const int k = 4 * g + e - HP - o + R;
          if (k >= 0 && k <= 2 * R) acc[o] = StencilOps<T>::mad(W.w[k], v[e], acc[o]);
        }
#pragma unroll
        for (int o = 0; o < O; o += 2) {  // (x[p], x[p+1]) -> (o, o+1): one FFMA2
          const int k = 4 * g + e - HP - o + R;
          if (k >= 0 && k <= 2 * R) fma2_into(acc[o], acc[o + 1], W.w[k], v[e], v[e + 1]);
        }
#pragma unroll
        for (int o = 0; o < O; o += 2) {  // x[p+1] -> even outputs (scalar)
          const int k = 4 * g + e + 1 - HP - o + R;
          if (k >= 0 && k <= 2 * R) acc[o] = StencilOps<T>::mad(W.w[k], v[e + 1], acc[o]);
        }
      }
    } else {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
#pragma unroll
        for (int o = 0; o < O; ++o) {
          const int k = 4 * g + e - HP - o + R;
          if (k >= 0 && k <= 2 * R) acc[o] = StencilOps<T>::mad(W.w[k], v[e], acc[o]);
        }
      }
    }
  }
  const long long cbase = c0 + sc0;
  if (cbase + O <= cols) {
    float* dst = orow + cbase;
    if constexpr (O % 8 == 0) {
#pragma unroll
      for (int q = 0; q < O / 8; ++q) {
        uint32_t raw[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) raw[e] = __float_as_uint(acc[8 * q + e]);
        st_stream<8>(dst + 8 * q, raw);
      }
    } else {
#pragma unroll
      for (int q = 0; q < O / 4; ++q) {
        uint32_t raw[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) raw[e] = __float_as_uint(acc[4 * q + e]);
        st_stream<4>(dst + 4 * q, raw);
      }
    }
  } else {
#pragma unroll
    for (int o = 0; o < O; ++o)
      if (cbase + o < cols) orow[cbase + o] = acc[o];
  }
}

template <int R, int O>
__global__ void __launch_bounds__(T1_THREADS)
overlap1d_tiled_kernel(const __grid_constant__ Weights1D W, int edge, float pad, const float* in, float* out,
                       size_t rows, size_t cols) {
  constexpr int TILE = T1_THREADS * O;  // outputs per tile
  extern __shared__ __align__(16) float sm[];
  const size_t tiles_per_row = (cols + TILE - 1) / TILE;
  const size_t ntiles = rows * tiles_per_row;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t row = tile / tiles_per_row;
    const long long c0 = static_cast<long long>((tile - row * tiles_per_row) * TILE);  // first output column
    stage_tile1<R, O, false>(sm, in + row * cols, (long long)cols, c0, edge, pad);
    __syncthreads();
    compute_tile1<R, O>(sm, W, out + row * cols, (long long)cols, c0);
    __syncthreads();  // the tile buffer is reused
  }
}

// Double-buffered persistent form ("_db"): while a block computes tile i from one buffer, the
// cp.async copies of tile i+1 fill the other. The (row, tile-in-row) coordinates advance by
// (G div tiles_per_row, G mod tiles_per_row) with one carry (no division per tile), and a tile whose
// halo lies inside its row is staged by a fast path: the addresses of a thread's 128-bit groups
// differ by compile-time constants, so a group costs one cp.async.
template <int R, int O, bool PK>
__global__ void __launch_bounds__(T1_THREADS)
overlap1d_tiled_db_kernel(const __grid_constant__ Weights1D W, int edge, float pad, const float* in, float* out,
                          size_t rows, size_t cols, unsigned buf_floats, unsigned tiles_per_row, unsigned dq, unsigned dr) {
  constexpr int TILE = T1_THREADS * O;
  constexpr int HP = (R + 3) / 4 * 4;
  constexpr int SPAN = TILE + 2 * HP;
  static_assert(O == 4 || 1024 % O == 0, "the padded layout must be linear in the group index");
  extern __shared__ __align__(16) float sm[];
  const size_t ntiles = rows * tiles_per_row;
  size_t tile = blockIdx.x;
  if (tile >= ntiles) return;
  size_t row = tile / tiles_per_row;                                  // the only division
  unsigned tcol = static_cast<unsigned>(tile - row * tiles_per_row);  // tile index inside the row
  auto advance = [&](size_t& t, size_t& r, unsigned& c) {
    t += gridDim.x;
    r += dq;
    c += dr;
    if (c >= tiles_per_row) {
      c -= tiles_per_row;
      ++r;
    }
  };
  const unsigned soff0 = static_cast<unsigned>(phys<O>(4 * threadIdx.x)) * 4u;  // byte offset of group t in a buffer
  constexpr unsigned SSTEP = (O == 4 ? 1024u : 1024u + 4096u / O) * 4u;          // ... of group t + 256
  auto stage = [&](size_t r, unsigned c, int b) {
    const long long c0 = static_cast<long long>(c) * TILE;
    const float* xrow = in + r * cols;
    float* dst = sm + size_t(b) * buf_floats;
    if (c0 - HP >= 0 && c0 + TILE + HP <= static_cast<long long>(cols)) {
      const float* g = xrow + c0 - HP + 4 * threadIdx.x;
      const uint32_t d = smem_u32(dst) + soff0;
#pragma unroll
      for (int k = 0; k < SPAN / 4 / T1_THREADS; ++k)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + k * SSTEP), "l"(g + k * 1024) : "memory");
      constexpr int KL = SPAN / 4 / T1_THREADS;  // the last, partial round of groups
      if (static_cast<int>(threadIdx.x) < SPAN / 4 - KL * T1_THREADS)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + KL * SSTEP), "l"(g + KL * 1024) : "memory");
    } else {
      stage_tile1<R, O, true>(dst, xrow, (long long)cols, c0, edge, pad);
    }
  };
  stage(row, tcol, 0);
  asm volatile("cp.async.commit_group;" ::: "memory");
  size_t ntile = tile, nrow = row;
  unsigned ntcol = tcol;
  advance(ntile, nrow, ntcol);
  int buf = 0;
  for (; tile < ntiles; buf ^= 1) {
    if (ntile < ntiles) stage(nrow, ntcol, buf ^ 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    __syncthreads();
    compute_tile1<R, O, PK>(sm + size_t(buf) * buf_floats, W, out + row * cols, (long long)cols,
                            static_cast<long long>(tcol) * TILE);
    __syncthreads();
    tile = ntile; row = nrow; tcol = ntcol;
    advance(ntile, nrow, ntcol);
  }
}

// ---- TMA-fed persistent form on a vector ("tma_swz_o16_s*") --------------------------------------
// The vector is viewed as a matrix of 128-byte rows (32 floats); one cp.async.bulk.tensor.2d per tile
// copies the TILE/32 + 2 rows around the tile (one whole row of halo on each side) into a stage in the
// 128-byte swizzle, which makes the 128-bit shared loads of threads 64 bytes apart conflict-free without
// padding. Completion is a `full` mbarrier per stage, reuse an `empty` one (one arrival per warp): no
// block barrier on the interior path and no staging instructions in the compute warps. Rows outside
// the vector arrive as zeros (CONSTANT-0); cells below 0, at or beyond floor(n / 32) * 32 (the ragged
// last row, which the tensor map cannot describe) or beyond n are patched in shared memory.
constexpr int T1W_TILE = T1_THREADS * 16;
constexpr int T1W_ROWS = T1W_TILE / 32 + 2;
constexpr unsigned T1W_STAGE_BYTES = T1W_ROWS * 128u;
constexpr unsigned T1W_STAGE_STRIDE = (T1W_STAGE_BYTES + 1023u) / 1024u * 1024u;

__device__ __forceinline__ void tma_load_rows(void* smem_dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(smem_dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar))
      : "memory");
}

template <int R, bool PK, int STAGES, typename T = float>
__global__ void __launch_bounds__(T1_THREADS)
overlap1d_tma_kernel(const __grid_constant__ Weights1D W, const __grid_constant__ CUtensorMap tmap, int edge, float pad,
                     const float* in, float* out, long long rows, long long cols, unsigned tiles_per_row, int ntiles,
                     unsigned* tile_ctr, unsigned tile_base) {
  constexpr int HP = (R + 3) / 4 * 4;
  constexpr int SWZ = (32 - HP) / 4;
  extern __shared__ unsigned char smraw0[];
  unsigned char* smraw = smraw0 + ((1024u - (smem_u32(smraw0) & 1023u)) & 1023u);  // the swizzle is a function of address bits 4..9
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw + STAGES * T1W_STAGE_STRIDE);
  uint64_t* empty = full + STAGES;
  int2* coord = reinterpret_cast<int2*>(empty + STAGES);  // (matrix row, tile column) of the tile in each stage; row < 0: end
  auto stage_ptr = [&](int s) { return reinterpret_cast<float*>(smraw + s * T1W_STAGE_STRIDE); };
  const int lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, T1_THREADS / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();
  const long long rows128 = cols >> 5;  // 128-byte rows per matrix row (rows > 1: cols % 32 == 0)
  // Dynamic tile assignment (see overlap2d_tiles.cuh "tma_*"): the first tile is the block's index, later ids come from
  // a global counter; the fetch is issued one tile ahead of its use; exactly one failing fetch per block.
  unsigned t_next = blockIdx.x;
  bool exhausted = false;
  auto produce = [&](int s) {  // thread 0
    const unsigned t = t_next;
    if (!exhausted) exhausted = t >= unsigned(ntiles);
    if (!exhausted) t_next = atomicAdd(tile_ctr, 1u) - tile_base + gridDim.x;
    if (!exhausted) {
      const unsigned prow = t / tiles_per_row, ptcol = t - prow * tiles_per_row;
      coord[s] = make_int2(int(prow), int(ptcol));
      mbar_arrive_expect_tx(full + s, T1W_STAGE_BYTES);
      tma_load_rows(stage_ptr(s), &tmap, 0, static_cast<int>(prow * rows128 + ptcol * (T1W_TILE / 32)) - 1, full + s);
    } else {
      coord[s] = make_int2(-1, 0);
      mbar_arrive(full + s);
    }
  };
  if (threadIdx.x == 0) {
#pragma unroll
    for (int d = 0; d < STAGES - 1; ++d) produce(d);
  }
  // Outside the vector the copy delivers zeros (what CONSTANT with pad 0 wants); outside a row of a matrix it delivers
  // the neighbouring rows. pb: the first column the 128-byte-row view does not hold as part of this row.
  const bool zeros_ok = rows == 1 && edge == EDGE_CONSTANT && bits_are_zero(pad);
  const long long pb = cols & ~31ll;
  const bool back_always = !zeros_ok || pb != cols;
  int s = 0, ph = 0;
  int tgt = STAGES - 1, tph = 1;
  for (int it = 0;; ++it) {
    if (threadIdx.x == 0) {
      if (it > 0) mbar_wait(empty + tgt, tph);
      produce(tgt);
    }
    tgt = tgt + 1 == STAGES ? 0 : tgt + 1;
    if (tgt == 0) tph ^= 1;
    mbar_wait(full + s, ph);
    const int2 rc = coord[s];
    if (rc.x < 0) break;
    const long long row = rc.x;
    const unsigned tcol = unsigned(rc.y);
    const long long c0 = static_cast<long long>(tcol) * T1W_TILE;
    float* sm = stage_ptr(s);
    const float* xrow = in + row * cols;
    auto put = [&](int idx, long long c) {  // window cell idx holds column c of the row
      const unsigned q = unsigned(idx) >> 5, ch = (unsigned(idx) >> 2) & 7u;
      sm[q * 32 + ((ch ^ (q & 7u)) << 2) + (idx & 3)] = ext_row(xrow, cols, c, edge, pad);
    };
    // Patches are per warp, not per block: only thread 0 reads the front halo, so warp 0 writes it; the cells from pb on
    // are written by every warp that gets here (same values), so no warp waits for another one.
    bool patched = false;
    if (tcol == 0 && !zeros_ok && threadIdx.x < 32) {
      put(lane, lane - 32);
      patched = true;
    }
    if (back_always && pb < c0 + T1W_TILE + 32) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const long long c = pb + lane + 32 * j;
        const long long idx = c - c0 + 32;
        if (idx < T1W_ROWS * 32) put(static_cast<int>(idx), c);
      }
      patched = true;
    }
    if (patched) {  // warp-uniform
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic writes before the next TMA refill
      __syncwarp();
    }
    compute_tile1<R, 16, PK, SWZ, T>(sm, W, out + row * cols, cols, c0);
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + s);
    s = s + 1 == STAGES ? 0 : s + 1;
    if (s == 0) ph ^= 1;
  }
}

// ---- register window + warp shuffles (no shared memory, no block barrier) ---------------------
// A thread owns 16 consecutive outputs: it fetches its own 16 inputs with two 256-bit loads (one
// full 32-byte sector each, all issued before the first use, like the Map kernel) and gets the r
// halo values on each side from the neighbouring lanes by shuffles; only lanes 0 and 31 read
// their outer halo from memory (those lines are being fetched by the neighbouring warp anyway).
template <int R, typename T = float>
__global__ void __launch_bounds__(T1_THREADS)
overlap1d_shfl_kernel(const __grid_constant__ Weights1D W, int edge, float pad, const float* in, float* out,
                      size_t rows, size_t cols) {
  constexpr int O = 16;
  constexpr int TILE = T1_THREADS * O;
  static_assert(R >= 1 && R <= O, "halo comes from the direct neighbours only");
  const int lane = threadIdx.x & 31;
  const size_t tiles_per_row = (cols + TILE - 1) / TILE;
  const size_t ntiles = rows * tiles_per_row;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t row = tile / tiles_per_row;
    const long long c0 = static_cast<long long>((tile - row * tiles_per_row) * TILE) + threadIdx.x * O;
    const float* x = in + row * cols;
    const long long lc = static_cast<long long>(cols);
    float win[O + 2 * R];
    if (c0 + O <= lc) {
      uint32_t a[8], b[8];
      ld_stream<8, true>(a, x + c0);
      ld_stream<8, true>(b, x + c0 + 8);
#pragma unroll
      for (int j = 0; j < 8; ++j) { win[R + j] = __uint_as_float(a[j]); win[R + 8 + j] = __uint_as_float(b[j]); }
    } else {
#pragma unroll
      for (int j = 0; j < O; ++j) win[R + j] = ext_row(x, lc, c0 + j, edge, pad);
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
      for (int j = 0; j < R; ++j) win[j] = ext_row(x, lc, c0 - R + j, edge, pad);
    }
    if (lane == 31) {
#pragma unroll
      for (int j = 0; j < R; ++j) win[R + O + j] = ext_row(x, lc, c0 + O + j, edge, pad);
    }
    float acc[O];
#pragma unroll
    for (int o = 0; o < O; ++o) acc[o] = 0.f;
    // Taps k with k - R even address window pairs (win[o+k], win[o+k+1]), o even, that are aligned
    // register pairs of the 256-bit loads: one FFMA2 per output pair (only worth it when the kernel
    // is issue bound, r >= 8). Per output the taps still accumulate in ascending k: bit-identical.
    constexpr bool PK = R >= 8 && StencilOps<T>::kFloat;
#pragma unroll
    for (int k = 0; k <= 2 * R; ++k) {
      if (PK && (k + R) % 2 == 0) {
#pragma unroll
        for (int o = 0; o < O; o += 2) fma2_into(acc[o], acc[o + 1], W.w[k], win[o + k], win[o + k + 1]);
      } else {
#pragma unroll
        for (int o = 0; o < O; ++o) acc[o] = StencilOps<T>::mad(W.w[k], win[o + k], acc[o]);
      }
    }
    if (c0 + O <= lc) {
      float* dst = out + row * cols + c0;
      uint32_t r0[8], r1[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) { r0[e] = __float_as_uint(acc[e]); r1[e] = __float_as_uint(acc[8 + e]); }
      st_stream<8>(dst, r0);
      st_stream<8>(dst + 8, r1);
    } else {
#pragma unroll
      for (int o = 0; o < O; ++o)
        if (c0 + o < lc) out[row * cols + c0 + o] = acc[o];
    }
  }
}

template <int R, typename T = float>
cudaError_t launch_shfl(const Launch& L, const Weights1D& w, int edge, float pad, const float* in, float* out,
                        size_t rows, size_t cols) {
  constexpr int TILE = T1_THREADS * 16;
  const size_t ntiles = rows * ((cols + TILE - 1) / TILE);
  const size_t grid = ntiles < 0x7fffffffu ? ntiles : 0x7fffffffu;
  overlap1d_shfl_kernel<R, T><<<(unsigned)grid, T1_THREADS, 0, L.stream>>>(w, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

// "regshfl_2x8": the same idea with warp-contiguous accesses. A warp owns 512 consecutive elements; lane l owns the
// two 8-element chunks A = [8l, 8l+8) and B = [256+8l, 256+8l+8) of them, so that each of the warp's two 256-bit
// loads (and stores) covers 1024 contiguous bytes (whole 128-byte lines, like the Map kernel) instead of every other
// 32-byte sector of 2048 bytes. Halos by shuffles with wrap-around: the right neighbour of lane 31's chunk A is lane
// 0's chunk B, the left neighbour of lane 0's chunk B is lane 31's chunk A; only A's left halo at lane 0 and B's right
// halo at lane 31 come from memory. r <= 8.
template <int R, typename T = float>
__global__ void __launch_bounds__(T1_THREADS)
overlap1d_shfl2_kernel(const __grid_constant__ Weights1D W, int edge, float pad, const float* in, float* out,
                       size_t rows, size_t cols) {
  constexpr int C = 8, TILE = T1_THREADS * 2 * C;
  static_assert(R >= 1 && R <= C, "halo comes from the direct neighbours only");
  constexpr unsigned FULLM = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t tiles_per_row = (cols + TILE - 1) / TILE;
  const size_t ntiles = rows * tiles_per_row;
  for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const size_t row = tile / tiles_per_row;
    const long long wbase = static_cast<long long>((tile - row * tiles_per_row) * TILE) + warp * (64 * C);
    const long long cA = wbase + C * lane, cB = cA + 32 * C;
    const float* x = in + row * cols;
    const long long lc = static_cast<long long>(cols);
    const bool full = wbase + 64 * C <= lc;  // warp-uniform
    float wa[C + 2 * R], wb[C + 2 * R];
    if (full) {
      uint32_t a[8], b[8];
      ld_stream<8, true>(a, x + cA);
      ld_stream<8, true>(b, x + cB);
#pragma unroll
      for (int j = 0; j < C; ++j) { wa[R + j] = __uint_as_float(a[j]); wb[R + j] = __uint_as_float(b[j]); }
    } else {
#pragma unroll
      for (int j = 0; j < C; ++j) {
        wa[R + j] = ext_row(x, lc, cA + j, edge, pad);
        wb[R + j] = ext_row(x, lc, cB + j, edge, pad);
      }
    }
    const int prev = (lane + 31) & 31, next = (lane + 1) & 31;
#pragma unroll
    for (int j = 0; j < R; ++j) {
      const float tA = __shfl_sync(FULLM, wa[C + j], prev);  // tail of the previous lane's A (lane 0: lane 31's)
      const float hA = __shfl_sync(FULLM, wa[R + j], next);  // head of the next lane's A
      const float tB = __shfl_sync(FULLM, wb[C + j], prev);
      const float hB = __shfl_sync(FULLM, wb[R + j], next);  // head of the next lane's B (lane 31: lane 0's)
      wa[j] = tA;                                  // lane 0: replaced below
      wa[R + C + j] = lane == 31 ? hB : hA;
      wb[j] = lane == 0 ? tA : tB;
      wb[R + C + j] = hB;                          // lane 31: replaced below
    }
    if (lane == 0) {
#pragma unroll
      for (int j = 0; j < R; ++j) wa[j] = ext_row(x, lc, cA - R + j, edge, pad);
    }
    if (lane == 31) {
#pragma unroll
      for (int j = 0; j < R; ++j) wb[R + C + j] = ext_row(x, lc, cB + C + j, edge, pad);
    }
    float accA[C], accB[C];
#pragma unroll
    for (int o = 0; o < C; ++o) accA[o] = accB[o] = 0.f;
    constexpr bool PK = R >= 8 && StencilOps<T>::kFloat;  // as in overlap1d_shfl_kernel: per output the taps accumulate in ascending k
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
          accA[o] = StencilOps<T>::mad(W.w[k], wa[o + k], accA[o]);
          accB[o] = StencilOps<T>::mad(W.w[k], wb[o + k], accB[o]);
        }
      }
    }
    float* orow = out + row * cols;
    if (full) {
      uint32_t r0[8], r1[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) { r0[e] = __float_as_uint(accA[e]); r1[e] = __float_as_uint(accB[e]); }
      st_stream<8>(orow + cA, r0);
      st_stream<8>(orow + cB, r1);
    } else {
#pragma unroll
      for (int o = 0; o < C; ++o) {
        if (cA + o < lc) orow[cA + o] = accA[o];
        if (cB + o < lc) orow[cB + o] = accB[o];
      }
    }
  }
}

template <int R, typename T = float>
cudaError_t launch_shfl2(const Launch& L, const Weights1D& w, int edge, float pad, const float* in, float* out,
                         size_t rows, size_t cols) {
  constexpr int TILE = T1_THREADS * 16;
  const size_t ntiles = rows * ((cols + TILE - 1) / TILE);
  const size_t grid = ntiles < 0x7fffffffu ? ntiles : 0x7fffffffu;
  overlap1d_shfl2_kernel<R, T><<<(unsigned)grid, T1_THREADS, 0, L.stream>>>(w, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

template <int O> constexpr size_t tiled_smem_bytes(int R) {
  const int HP = (R + 3) / 4 * 4;
  const int span = T1_THREADS * O + 2 * HP;
  return size_t(O == 4 ? span : span + 4 * (span / O) + 4) * sizeof(float);
}

struct O1Variant { const char* name; int o; };  // o == 0: direct
const O1Variant kVariants[] = {{"direct", 0}, {"tiled_o4", 4}, {"tiled_o8", 8}, {"tiled_o16", 16}, {"regshfl_o16", -16},
                               {"tiled_o8_db", 108}, {"tiled_o16_db", 116}, {"tiled_o16_db_ffma2", 216},
                               {"regshfl_2x8", -8}, {"tma_swz_o16_s2", 302}, {"tma_swz_o16_s3", 303}};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

inline bool templated_radius(int r) { return r == 1 || r == 2 || r == 3 || r == 4 || r == 8 || r == 16; }

template <int R, int O>
cudaError_t launch_tiled(const Launch& L, const Weights1D& w, int edge, float pad, const float* in, float* out,
                         size_t rows, size_t cols) {
  constexpr int TILE = T1_THREADS * O;
  const size_t smem = tiled_smem_bytes<O>(R);
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(overlap1d_tiled_kernel<R, O>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_done = true;
  }
  const size_t ntiles = rows * ((cols + TILE - 1) / TILE);
  size_t grid = ntiles < 0x7fffffffu ? ntiles : 0x7fffffffu;
  overlap1d_tiled_kernel<R, O><<<(unsigned)grid, T1_THREADS, smem, L.stream>>>(w, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

template <int R, int O, bool PK>
cudaError_t launch_tiled_db(const Launch& L, const Weights1D& w, int edge, float pad, const float* in, float* out,
                            size_t rows, size_t cols) {
  constexpr int TILE = T1_THREADS * O;
  const size_t one = (tiled_smem_bytes<O>(R) + 15) / 16 * 16;
  const size_t smem = 2 * one;
  auto kern = overlap1d_tiled_db_kernel<R, O, PK>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T1_THREADS, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  const size_t ntiles = rows * ((cols + TILE - 1) / TILE);
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  const size_t tpr = (cols + TILE - 1) / TILE;
  if (tpr >= (size_t(1) << 31)) return cudaErrorInvalidValue;
  kern<<<(unsigned)grid, T1_THREADS, smem, L.stream>>>(w, edge, pad, in, out, rows, cols, (unsigned)(one / 4), (unsigned)tpr,
                                                        (unsigned)(grid / tpr), (unsigned)(grid % tpr));
  ++*L.launches;
  return cudaGetLastError();
}

// Tensor map of a vector seen as floor(n / 32) rows of 32 floats, box = 32 x T1W_ROWS, 128-byte swizzle (host side;
// the driver entry point is looked up through the runtime, libcuda is not linked). The last map is cached.
inline cudaError_t make_tmap_rows(CUtensorMap* out, const float* base, size_t nrows) {
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
  static thread_local const float* last_base = nullptr;
  static thread_local size_t last_rows = 0;
  static thread_local CUtensorMap last_map;
  if (last_base == base && last_rows == nrows) {
    *out = last_map;
    return cudaSuccess;
  }
  const cuuint64_t dims[2] = {32, nrows};
  const cuuint64_t strides[1] = {128};
  const cuuint32_t box[2] = {32, cuuint32_t(T1W_ROWS)};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  last_base = base;
  last_rows = nrows;
  last_map = *out;
  return cudaSuccess;
}

// vectors shorter than one tile (and anything the tensor map cannot describe) take the cp.async form
template <int R, int STAGES, typename T = float>
cudaError_t launch_tma1(const Launch& L, const Weights1D& w, int edge, float pad, const float* in, float* out, size_t rows,
                        size_t cols) {
  const size_t tpr = (cols + T1W_TILE - 1) / T1W_TILE;
  const size_t ntiles = rows * tpr;
  if ((rows == 1 && cols < size_t(T1W_TILE)) || cols < 32 || rows * cols / 32 >= (size_t(1) << 31) - 1 || ntiles >= (size_t(1) << 30)) {
    if constexpr (StencilOps<T>::kFloat) return launch_tiled_db<R, 16, true>(L, w, edge, pad, in, out, rows, cols);
    else return launch_shfl<R, T>(L, w, edge, pad, in, out, rows, cols);
  }
  constexpr size_t smem = size_t(STAGES) * T1W_STAGE_STRIDE + 3 * STAGES * sizeof(uint64_t) + 1024;  // stages, full/empty, coord
  auto kern = overlap1d_tma_kernel<R, true, STAGES, T>;
  static int per_sm = 0;
  if (per_sm == 0) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T1_THREADS, smem) != cudaSuccess || per_sm < 1)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tmap;
  cudaError_t e = make_tmap_rows(&tmap, in, rows * cols / 32);
  if (e != cudaSuccess) return e;
  size_t grid = size_t(L.sms) * per_sm;
  if (grid > ntiles) grid = ntiles;
  kern<<<(unsigned)grid, T1_THREADS, smem, L.stream>>>(w, tmap, edge, pad, in, out, (long long)rows, (long long)cols,
                                                        (unsigned)tpr, (int)ntiles, L.tile_ctr, *L.tile_next);
  *L.tile_next += unsigned(ntiles);  // ntiles - grid ids fetched from the counter + one failing fetch per block
  ++*L.launches;
  return cudaGetLastError();
}

template <int STAGES, typename T = float>
cudaError_t launch_tma1_r(const Launch& L, const Weights1D& w, int r, int edge, float pad, const float* in, float* out,
                          size_t rows, size_t cols) {
  switch (r) {
    case 1: return launch_tma1<1, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
    case 2: return launch_tma1<2, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
    case 3: return launch_tma1<3, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
    case 4: return launch_tma1<4, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
    case 8: return launch_tma1<8, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
    case 16: return launch_tma1<16, STAGES, T>(L, w, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

// int32 elements (reading 26): the direct, register-window and TMA-fed variants
cudaError_t launch_overlap1d_rows_i32(const Launch& L, int o, const Weights1D& w, int r, int edge, float pad,
                                      const float* in, float* out, size_t rows, size_t cols) {
  using T = int32_t;
  switch (o) {
    case 0: {
      const size_t total = rows * cols;
      size_t grid = (total + 255) / 256;
      const size_t cap = size_t(L.sms) * 64;
      if (grid > cap) grid = cap;
      overlap1d_direct_kernel<T><<<(unsigned)grid, 256, 0, L.stream>>>(w, r, edge, pad, in, out, rows, cols);
      ++*L.launches;
      return cudaGetLastError();
    }
    case 302: return launch_tma1_r<2, T>(L, w, r, edge, pad, in, out, rows, cols);
    case 303: return launch_tma1_r<3, T>(L, w, r, edge, pad, in, out, rows, cols);
    case -8:
      switch (r) {
        case 1: return launch_shfl2<1, T>(L, w, edge, pad, in, out, rows, cols);
        case 2: return launch_shfl2<2, T>(L, w, edge, pad, in, out, rows, cols);
        case 3: return launch_shfl2<3, T>(L, w, edge, pad, in, out, rows, cols);
        case 4: return launch_shfl2<4, T>(L, w, edge, pad, in, out, rows, cols);
        case 8: return launch_shfl2<8, T>(L, w, edge, pad, in, out, rows, cols);
      }
      return cudaErrorInvalidValue;
    case -16:
      switch (r) {
        case 1: return launch_shfl<1, T>(L, w, edge, pad, in, out, rows, cols);
        case 2: return launch_shfl<2, T>(L, w, edge, pad, in, out, rows, cols);
        case 3: return launch_shfl<3, T>(L, w, edge, pad, in, out, rows, cols);
        case 4: return launch_shfl<4, T>(L, w, edge, pad, in, out, rows, cols);
        case 8: return launch_shfl<8, T>(L, w, edge, pad, in, out, rows, cols);
        case 16: return launch_shfl<16, T>(L, w, edge, pad, in, out, rows, cols);
      }
      return cudaErrorInvalidValue;
  }
  return cudaErrorInvalidValue;
}

template <int O, bool PK>
cudaError_t launch_tiled_db_r(const Launch& L, const Weights1D& w, int r, int edge, float pad, const float* in,
                              float* out, size_t rows, size_t cols) {
  switch (r) {
    case 1: return launch_tiled_db<1, O, PK>(L, w, edge, pad, in, out, rows, cols);
    case 2: return launch_tiled_db<2, O, PK>(L, w, edge, pad, in, out, rows, cols);
    case 3: return launch_tiled_db<3, O, PK>(L, w, edge, pad, in, out, rows, cols);
    case 4: return launch_tiled_db<4, O, PK>(L, w, edge, pad, in, out, rows, cols);
    case 8: return launch_tiled_db<8, O, PK>(L, w, edge, pad, in, out, rows, cols);
    case 16: return launch_tiled_db<16, O, PK>(L, w, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

template <int O>
cudaError_t launch_tiled_r(const Launch& L, const Weights1D& w, int r, int edge, float pad, const float* in,
                           float* out, size_t rows, size_t cols) {
  switch (r) {
    case 1: return launch_tiled<1, O>(L, w, edge, pad, in, out, rows, cols);
    case 2: return launch_tiled<2, O>(L, w, edge, pad, in, out, rows, cols);
    case 3: return launch_tiled<3, O>(L, w, edge, pad, in, out, rows, cols);
    case 4: return launch_tiled<4, O>(L, w, edge, pad, in, out, rows, cols);
    case 8: return launch_tiled<8, O>(L, w, edge, pad, in, out, rows, cols);
    case 16: return launch_tiled<16, O>(L, w, edge, pad, in, out, rows, cols);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

int overlap1d_variant_count() { return kNumVariants; }
const char* overlap1d_variant_name(int v) { return (v >= 0 && v < kNumVariants) ? kVariants[v].name : nullptr; }

bool overlap1d_variant_ok(int v, int dtype, int r, const void* in, const void* out, size_t rows, size_t cols) {
  if (v < 0 || v >= kNumVariants) return false;
  if (kVariants[v].o == 0) return true;
  if (dtype != DT_F32 && kVariants[v].o > 0 && kVariants[v].o < 300) return false;  // i32: direct, regshfl_*, tma_* only
  if (r < 0 || r > 16) return false;  // radii between the instantiated ones run zero-padded (kernels.hpp)
  if (kVariants[v].o == -8 && r > 8) return false;
  if (kVariants[v].o >= 300 && rows != 1 && cols % 32 != 0) return false;  // a matrix row must be whole 128-byte rows
  const bool al = reinterpret_cast<uintptr_t>(in) % 32 == 0 && reinterpret_cast<uintptr_t>(out) % 32 == 0;
  return al && (rows == 1 || cols % 8 == 0);
}

cudaError_t launch_overlap1d_rows(const Launch& L, int v, int dtype, const Weights1D& w, int r, int edge, float pad,
                                  const float* in, float* out, size_t rows, size_t cols) {
  if (rows * cols == 0) return cudaSuccess;
  if (kVariants[v].o != 0 && !templated_radius(r)) {
    const int R = padded_radius_1d(r);
    if (R < 0) return cudaErrorInvalidValue;
    return launch_overlap1d_rows(L, v, dtype, pad_weights_1d(w, r, R), R, edge, pad, in, out, rows, cols);
  }
  if (dtype != DT_F32) return launch_overlap1d_rows_i32(L, kVariants[v].o, w, r, edge, pad, in, out, rows, cols);
  switch (kVariants[v].o) {
    case 0: {
      const size_t total = rows * cols;
      size_t grid = (total + 255) / 256;
      const size_t cap = size_t(L.sms) * 64;
      if (grid > cap) grid = cap;
      overlap1d_direct_kernel<float><<<(unsigned)grid, 256, 0, L.stream>>>(w, r, edge, pad, in, out, rows, cols);
      ++*L.launches;
      return cudaGetLastError();
    }
    case 4: return launch_tiled_r<4>(L, w, r, edge, pad, in, out, rows, cols);
    case 8: return launch_tiled_r<8>(L, w, r, edge, pad, in, out, rows, cols);
    case 16: return launch_tiled_r<16>(L, w, r, edge, pad, in, out, rows, cols);
    case 108: return launch_tiled_db_r<8, false>(L, w, r, edge, pad, in, out, rows, cols);
    case 116: return launch_tiled_db_r<16, false>(L, w, r, edge, pad, in, out, rows, cols);
    case 216: return launch_tiled_db_r<16, true>(L, w, r, edge, pad, in, out, rows, cols);
    case 302: return launch_tma1_r<2>(L, w, r, edge, pad, in, out, rows, cols);
    case 303: return launch_tma1_r<3>(L, w, r, edge, pad, in, out, rows, cols);
    case -8:
      switch (r) {
        case 1: return launch_shfl2<1>(L, w, edge, pad, in, out, rows, cols);
        case 2: return launch_shfl2<2>(L, w, edge, pad, in, out, rows, cols);
        case 3: return launch_shfl2<3>(L, w, edge, pad, in, out, rows, cols);
        case 4: return launch_shfl2<4>(L, w, edge, pad, in, out, rows, cols);
        case 8: return launch_shfl2<8>(L, w, edge, pad, in, out, rows, cols);
      }
      return cudaErrorInvalidValue;
    case -16:
      switch (r) {
        case 1: return launch_shfl<1>(L, w, edge, pad, in, out, rows, cols);
        case 2: return launch_shfl<2>(L, w, edge, pad, in, out, rows, cols);
        case 3: return launch_shfl<3>(L, w, edge, pad, in, out, rows, cols);
        case 4: return launch_shfl<4>(L, w, edge, pad, in, out, rows, cols);
        case 8: return launch_shfl<8>(L, w, edge, pad, in, out, rows, cols);
        case 16: return launch_shfl<16>(L, w, edge, pad, in, out, rows, cols);
      }
      return cudaErrorInvalidValue;
  }
  return cudaErrorInvalidValue;
}

}  // namespace skel
