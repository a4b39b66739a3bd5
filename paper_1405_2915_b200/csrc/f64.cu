// fp64 elements ("f64 element types for all skeletons"; reading 27): one kernel per
// skeleton, the streaming structure of the f32 / i32 kernels without their variant tables.
//   Map / three-vector Map   256-bit accesses (4 doubles), two vectors per operand in flight, one block per tile;
//                            add / mult correctly rounded, saxpy and muladd ONE fused multiply-add (DFMA).
//   Reduce / MapReduce       one block per contiguous chunk (hardware-balanced), 4 accumulators per thread, fixed
//                            shuffle + shared-memory trees, last block (ticket) folds the partials in index order:
//                            bitwise deterministic for a given n, no floating-point atomics.
//   Scan                     n >= 2^20: ONE pass over HBM ("l2ahead": a reduce pass runs two tiles ahead and publishes
//                            tile aggregates, the scan pass re-reads the tile from L2; 16 B/elem of HBM traffic);
//                            smaller n: three kernels in a fixed order (chunk totals, exclusive scan of the totals
//                            by one block, chunk-local scans with their offsets). Both deterministic run to run.
//   MapOverlap 1D / 2D       one output per thread, taps in ascending order, one DFMA each; chains of at most 33 taps
//                            (2D: one chain per filter row, the row sums added): bound 33 * 2^-53 of sum|w x|.
// All of them are bound by HBM (fp64 arithmetic is far from its limit at these intensities).
#include "common.cuh"
#include "kernels.hpp"

namespace skel {
namespace {

enum : int { EDGE_CONSTANT = 0, EDGE_DUPLICATE = 1, EDGE_CYCLIC = 2 };
constexpr int D_THREADS = 256;

template <int FN> __device__ __forceinline__ double dapply(double c, double a, double b) {
  if constexpr (FN == FN_ADD) return __dadd_rn(a, b);
  else if constexpr (FN == FN_MULT) return __dmul_rn(a, b);
  else if constexpr (FN == FN_MAX) return a < b ? b : a;
  else if constexpr (FN == FN_SAXPY) return __fma_rn(c, a, b);
  else return a;  // FN_IDENT
}
template <int OP> __device__ __forceinline__ double didentity() {
  if constexpr (OP == FN_ADD) return 0.0;
  else if constexpr (OP == FN_MULT) return 1.0;
  else return -INFINITY;
}
template <int OP> __device__ __forceinline__ double dwarp_reduce(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = dapply<OP>(0.0, v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// block-wide reduction in a fixed order; result valid in thread 0; smem holds 32 doubles
template <int OP> __device__ __forceinline__ double dblock_reduce(double v, double* smem) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  v = dwarp_reduce<OP>(v);
  if (lane == 0) smem[warp] = v;
  __syncthreads();
  if (warp == 0) {
    v = lane < D_THREADS / 32 ? smem[lane] : didentity<OP>();
    v = dwarp_reduce<OP>(v);
  }
  return v;
}

__device__ __forceinline__ void ld4(double (&d)[4], const double* p) {  // 256-bit load, L1 no-allocate
  uint32_t r[8];
  ld_stream<8, false>(r, p);
#pragma unroll
  for (int j = 0; j < 4; ++j) d[j] = __hiloint2double(static_cast<int>(r[2 * j + 1]), static_cast<int>(r[2 * j]));
}
__device__ __forceinline__ void st4(double* p, const double (&d)[4]) {
  uint32_t r[8];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    r[2 * j] = static_cast<uint32_t>(__double2loint(d[j]));
    r[2 * j + 1] = static_cast<uint32_t>(__double2hiint(d[j]));
  }
  st_stream<8>(p, r);
}

// ---- Map ------------------------------------------------------------------------------------------------------
// NIN = 1: out = f(in0, c); 2: out = f(in0, in1); 3: out = in0 * in1 + in2 (MULADD). Every element is read and
// written by the same thread, so `out` may alias any input.
template <int FN, int NIN>
__global__ void __launch_bounds__(D_THREADS)
map_f64_kernel(double c, const double* in0, const double* in1, const double* in2, double* out, size_t n) {
  constexpr int U = 2;
  const size_t base = (size_t(blockIdx.x) * U * D_THREADS + threadIdx.x) * 4;
  const bool vec_ok = (reinterpret_cast<uintptr_t>(in0) | reinterpret_cast<uintptr_t>(out) |
                       (NIN >= 2 ? reinterpret_cast<uintptr_t>(in1) : 0) | (NIN >= 3 ? reinterpret_cast<uintptr_t>(in2) : 0)) % 32 == 0;
  if (vec_ok && base + size_t(U - 1) * D_THREADS * 4 + 4 <= n) {
    double a[U][4], b[U][4], d[U][4];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      ld4(a[u], in0 + base + size_t(u) * D_THREADS * 4);
      if (NIN >= 2) ld4(b[u], in1 + base + size_t(u) * D_THREADS * 4);
      if (NIN >= 3) ld4(d[u], in2 + base + size_t(u) * D_THREADS * 4);
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      double r[4];
#pragma unroll
      for (int j = 0; j < 4; ++j)
        r[j] = NIN == 3 ? __fma_rn(a[u][j], b[u][j], d[u][j]) : dapply<FN>(c, a[u][j], NIN == 2 ? b[u][j] : c);
      st4(out + base + size_t(u) * D_THREADS * 4, r);
    }
  } else {
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const size_t i = base + size_t(u) * D_THREADS * 4 + j;
        if (i < n) out[i] = NIN == 3 ? __fma_rn(in0[i], in1[i], in2[i]) : dapply<FN>(c, in0[i], NIN == 2 ? in1[i] : c);
      }
  }
}

// ---- Reduce / MapReduce -----------------------------------------------------------------------------------------
// FOLD = false: only the chunk totals are wanted (partials[b], phase 1 of the Scan); no ticket, no fold.
template <int MAPF, bool HAS_IN1, int OP, bool FOLD = true>
__global__ void __launch_bounds__(D_THREADS)
mapreduce_f64_kernel(const double* in0, const double* in1, double c, size_t n, size_t chunk, double* partials,
                     unsigned* ticket, double* result) {
  __shared__ double smem[32];
  __shared__ bool is_last;
  const size_t lo = size_t(blockIdx.x) * chunk, hi = lo + chunk < n ? lo + chunk : n;
  double acc[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) acc[j] = didentity<OP>();
  const bool vec_ok = (reinterpret_cast<uintptr_t>(in0) | (HAS_IN1 ? reinterpret_cast<uintptr_t>(in1) : 0)) % 32 == 0;
  size_t i = lo + size_t(threadIdx.x) * 4;  // chunk is a multiple of 4 * D_THREADS: every block starts aligned
  for (; i + 4 <= hi; i += size_t(D_THREADS) * 4) {
    double a[4], b[4];
    if (vec_ok) {
      ld4(a, in0 + i);
      if (HAS_IN1) ld4(b, in1 + i);
    } else {  // operands not 32-byte aligned (adopted buffers)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        a[j] = in0[i + j];
        if (HAS_IN1) b[j] = in1[i + j];
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[j] = dapply<OP>(0.0, acc[j], dapply<MAPF>(c, a[j], HAS_IN1 ? b[j] : c));
  }
  for (int j = 0; j < 4; ++j)  // the ragged last group of the vector (at most one thread has one)
    if (i + j < hi) acc[j] = dapply<OP>(0.0, acc[j], dapply<MAPF>(c, in0[i + j], HAS_IN1 ? in1[i + j] : c));
  double v = dapply<OP>(0.0, dapply<OP>(0.0, acc[0], acc[1]), dapply<OP>(0.0, acc[2], acc[3]));
  v = dblock_reduce<OP>(v, smem);
  if constexpr (!FOLD) {
    if (threadIdx.x == 0) partials[blockIdx.x] = v;
    return;
  }
  if (gridDim.x == 1) {
    if (threadIdx.x == 0) *result = v;
    return;
  }
  if (threadIdx.x == 0) {
    partials[blockIdx.x] = v;
    __threadfence();
    const unsigned t = atomicInc(ticket, gridDim.x - 1);
    is_last = t == gridDim.x - 1;
  }
  __syncthreads();
  if (is_last) {
    __threadfence();
    double a = didentity<OP>();
    for (unsigned k = threadIdx.x; k < gridDim.x; k += D_THREADS) a = dapply<OP>(0.0, a, partials[k]);
    __syncthreads();
    a = dblock_reduce<OP>(a, smem);
    if (threadIdx.x == 0) *result = a;
  }
}

// ---- Scan ---------------------------------------------------------------------------------------------------------
// block-wide exclusive prefix of one value per thread in thread order, plus the block total (both in fixed order)
template <int OP>
__device__ __forceinline__ double dblock_exclusive(double v, double* smem, double* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc = dapply<OP>(0.0, t, inc);
  }
  if (lane == 31) smem[warp] = inc;
  __syncthreads();
  double wprefix = didentity<OP>(), tot = didentity<OP>();
#pragma unroll
  for (int w = 0; w < D_THREADS / 32; ++w) {
    const double s = smem[w];
    if (w < warp) wprefix = dapply<OP>(0.0, wprefix, s);
    tot = dapply<OP>(0.0, tot, s);
  }
  __syncthreads();  // smem is reused by the next call
  double exc = __shfl_up_sync(0xffffffffu, inc, 1);
  if (lane == 0) exc = didentity<OP>();
  *total = tot;
  return dapply<OP>(0.0, wprefix, exc);
}

// phase 1: total of every chunk (the Reduce kernel with FN_IDENT writes partials[b]); phase 2:
template <int OP>
__global__ void __launch_bounds__(D_THREADS) scan_f64_offsets_kernel(double* partials, unsigned nchunks, double init) {
  __shared__ double smem[32];
  // one block scans the chunk totals in index order: partials[b] becomes init (+) total of the chunks before b
  double carry = init;
  for (unsigned base = 0; base < nchunks; base += D_THREADS) {
    const unsigned k = base + threadIdx.x;
    const double v = k < nchunks ? partials[k] : didentity<OP>();
    double tot;
    const double exc = dblock_exclusive<OP>(v, smem, &tot);
    if (k < nchunks) partials[k] = dapply<OP>(0.0, carry, exc);
    carry = dapply<OP>(0.0, carry, tot);
  }
}

// phase 3: the scan of chunk b, started from its offset
template <int OP, bool EXCLUSIVE>
__global__ void __launch_bounds__(D_THREADS)
scan_f64_apply_kernel(const double* in, double* out, size_t n, size_t chunk, const double* offsets) {
  __shared__ double smem[32];
  const size_t lo = size_t(blockIdx.x) * chunk, hi = lo + chunk < n ? lo + chunk : n;
  double carry = offsets[blockIdx.x];
  for (size_t base = lo; base < hi; base += size_t(D_THREADS) * 4) {
    const size_t i = base + size_t(threadIdx.x) * 4;
    const bool vec = i + 4 <= hi && (reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) % 32 == 0;
    double x[4];
    if (vec) ld4(x, in + i);
    else {
#pragma unroll
      for (int j = 0; j < 4; ++j) x[j] = i + j < hi ? in[i + j] : didentity<OP>();
    }
    double tsum = x[0];
#pragma unroll
    for (int j = 1; j < 4; ++j) tsum = dapply<OP>(0.0, tsum, x[j]);
    double tot;
    double run = dapply<OP>(0.0, carry, dblock_exclusive<OP>(tsum, smem, &tot));
    double y[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const double before = run;
      run = dapply<OP>(0.0, run, x[j]);
      y[j] = EXCLUSIVE ? before : run;
    }
    if (vec) st4(out + i, y);
    else {
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i + j < hi) out[i + j] = y[j];
    }
    carry = dapply<OP>(0.0, carry, tot);
  }
}

// ---- MapOverlap ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ long long wrap_index(long long j, long long n, int edge) {  // j outside [0, n), not CONSTANT
  if (edge == EDGE_CYCLIC) {
    const long long m = j % n;
    return m < 0 ? m + n : m;
  }
  return j < 0 ? 0 : n - 1;
}

// 1D on a vector (rows = 1) or along the rows (axis 0) / columns (axis 1) of a matrix. A thread owns 4 consecutive
// elements of a matrix row (a warp's accesses stay coalesced for both axes). Row-wise, r <= 16, interior: the 4 outputs share a window of 4 + 2r values,
// each loaded once and used for up to 4 taps (taps still ascend per output). Everything else: one output at a time.
__device__ __forceinline__ double overlap1d_f64_one(const Weights1D64& W, int r, int edge, double pad, const double* line,
                                                    long long len, long long stride, long long pos) {
  const int chain = 2 * r + 1 <= 33 ? 33 : 16;
  double total_acc = 0.0;
  for (int k0 = 0; k0 <= 2 * r; k0 += chain) {
    const int k1 = k0 + chain < 2 * r + 1 ? k0 + chain : 2 * r + 1;
    double acc = 0.0;
    for (int k = k0; k < k1; ++k) {
      const long long q = pos + k - r;
      double v;
      if (q >= 0 && q < len) v = __ldg(line + q * stride);
      else if (edge == EDGE_CONSTANT) v = pad;
      else v = __ldg(line + wrap_index(q, len, edge) * stride);
      acc = __fma_rn(W.w[k], v, acc);
    }
    total_acc = k0 == 0 ? acc : __dadd_rn(total_acc, acc);
  }
  return total_acc;
}

__global__ void __launch_bounds__(D_THREADS)
overlap1d_f64_kernel(const __grid_constant__ Weights1D64 W, int r, int edge, double pad, int axis, const double* in,
                     double* out, size_t rows, size_t cols) {
  const size_t groups_per_row = (cols + 3) / 4, ngroups = rows * groups_per_row;
  const long long lr = static_cast<long long>(rows), lc = static_cast<long long>(cols);
  for (size_t g = blockIdx.x * size_t(D_THREADS) + threadIdx.x; g < ngroups; g += size_t(gridDim.x) * D_THREADS) {
    const long long i = static_cast<long long>(g / groups_per_row), j0 = static_cast<long long>(g - size_t(i) * groups_per_row) * 4;
    double* dst = out + size_t(i) * cols + j0;
    if (axis == 0 && r <= 16 && j0 - r >= 0 && j0 + 3 + r < lc) {  // interior of a row: shared window
      const double* x = in + size_t(i) * cols + j0 - r;
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      for (int t = 0; t < 4 + 2 * r; ++t) {
        const double v = __ldg(x + t);
#pragma unroll
        for (int o = 0; o < 4; ++o) {
          const int k = t - o;
          if (k >= 0 && k <= 2 * r) acc[o] = __fma_rn(W.w[k], v, acc[o]);
        }
      }
#pragma unroll
      for (int o = 0; o < 4; ++o) dst[o] = acc[o];
    } else {
      for (int o = 0; o < 4 && j0 + o < lc; ++o)
        dst[o] = axis == 0 ? overlap1d_f64_one(W, r, edge, pad, in + size_t(i) * cols, lc, 1, j0 + o)
                           : overlap1d_f64_one(W, r, edge, pad, in + j0 + o, lr, lc, i);
    }
  }
}

// Row-wise fast form, radius <= R (the weights arrive zero-padded to 2R+1 taps: a zero weight adds exactly 0, the taps
// keep their ascending order, reading 28): a thread owns 4 consecutive outputs, reads its 4 + 2R window with
// 1 + R/2 aligned 256-bit loads (the scalar form above needs 4 + 2R 8-byte loads, and the L1 tag stage, not HBM, is
// what bounds it) and stores one 256-bit vector; all taps unrolled, weights straight from the constant bank. Groups
// whose window leaves the row take the per-element path. Needs 32-byte aligned rows: base pointers and cols % 4 == 0.
__device__ __forceinline__ void ld4_cached(double (&d)[4], const double* p) {  // 256-bit read-only load that allocates in
  uint32_t r[8];                                                              // L1: neighbours re-read the window
  asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "l"(p));
#pragma unroll
  for (int j = 0; j < 4; ++j) d[j] = __hiloint2double(static_cast<int>(r[2 * j + 1]), static_cast<int>(r[2 * j]));
}

template <int R>
__global__ void __launch_bounds__(D_THREADS)
overlap1d_f64_rows_kernel(const __grid_constant__ Weights1D64 W, int r_true, int edge, double pad, const double* in,
                          double* out, size_t rows, size_t cols) {
  const size_t groups_per_row = cols / 4, ngroups = rows * groups_per_row;
  const long long lc = static_cast<long long>(cols);
  for (size_t g = blockIdx.x * size_t(D_THREADS) + threadIdx.x; g < ngroups; g += size_t(gridDim.x) * D_THREADS) {
    const size_t i = g / groups_per_row;
    const long long j0 = static_cast<long long>(g - i * groups_per_row) * 4;
    const double* row = in + i * cols;
    double* dst = out + i * cols + j0;
    if (j0 - R >= 0 && j0 + 3 + R < lc) {
      double v[4 + 2 * R];
#pragma unroll
      for (int c = 0; c < 1 + R / 2; ++c) ld4_cached(*reinterpret_cast<double(*)[4]>(v + 4 * c), row + j0 - R + 4 * c);
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int k = 0; k <= 2 * R; ++k)
#pragma unroll
        for (int o = 0; o < 4; ++o) acc[o] = __fma_rn(W.w[k], v[o + k], acc[o]);
      st4(dst, acc);
    } else {  // the true radius and the unpadded taps sit in the middle of W
      for (int o = 0; o < 4; ++o) {
        double a = 0.0;
        for (int k = 0; k <= 2 * r_true; ++k) {
          long long q = j0 + o + k - r_true;
          double x;
          if (q < 0 || q >= lc) {
            if (edge == EDGE_CONSTANT) x = pad;
            else x = row[wrap_index(q, lc, edge)];
          } else x = row[q];
          a = __fma_rn(W.w[k + R - r_true], x, a);
        }
        dst[o] = a;
      }
    }
  }
}

__global__ void __launch_bounds__(D_THREADS)
overlap2d_f64_kernel(const __grid_constant__ Weights2D64 W, int ry, int rx, int edge, double pad, const double* in,
                     double* out, size_t rows, size_t cols) {
  const size_t total = rows * cols;
  const int fw = 2 * rx + 1;
  const long long lr = static_cast<long long>(rows), lc = static_cast<long long>(cols);
  for (size_t idx = blockIdx.x * size_t(D_THREADS) + threadIdx.x; idx < total; idx += size_t(gridDim.x) * D_THREADS) {
    const long long i = static_cast<long long>(idx / cols), j = static_cast<long long>(idx - size_t(i) * cols);
    double acc = 0.0;
    for (int a = 0; a <= 2 * ry; ++a) {  // one chain per filter row, the row sums added
      long long p = i + a - ry;
      const bool p_out = p < 0 || p >= lr;
      if (p_out && edge != EDGE_CONSTANT) p = wrap_index(p, lr, edge);
      double s = 0.0;
      for (int b = 0; b <= 2 * rx; ++b) {
        long long q = j + b - rx;
        const bool q_out = q < 0 || q >= lc;
        double v;
        if ((p_out || q_out) && edge == EDGE_CONSTANT) v = pad;
        else {
          if (q_out) q = wrap_index(q, lc, edge);
          v = __ldg(in + p * lc + q);
        }
        s = __fma_rn(W.w[a * fw + b], v, s);
      }
      acc = a == 0 ? s : __dadd_rn(acc, s);
    }
    out[idx] = acc;
  }
}

// ---- Scan, single pass over HBM ("l2ahead", the structure of scan.cu's scan_l2_kernel for 8-byte elements) ------------
// CTA b owns tiles b, b + G, ... (static, cooperative launch). Worker warps: a ring of S bulk async copies (evict_last)
// feeds a REDUCE pass that runs D tiles ahead and publishes each tile's aggregate; the SCAN pass re-reads the tile (an
// L2 hit), scans it in registers, adds the carry and streams it out. One PREFIX warp per CTA computes the carry of the
// CTA's next tile as the carry of its previous tile (+) the G aggregates in between, all loads of the window in flight.
// A tile's state is 16 bytes, (aggregate bits, launch number), written and read with ONE 128-bit relaxed.gpu access
// (single-copy atomic): a reader that sees this launch's number sees this launch's aggregate. The launch number never
// repeats (64 bits), so the array is never cleared. The grouping of every sum depends on (n, G) only: bitwise
// deterministic run to run on a given GPU, like the three-kernel form (whose rounding it does not share).
__device__ __forceinline__ void ld_state128(const unsigned long long* p, unsigned long long& value, unsigned long long& tag) {
  asm volatile("{\n.reg .b128 t;\nld.relaxed.gpu.global.b128 t, [%2];\nmov.b128 {%0, %1}, t;\n}"
               : "=l"(value), "=l"(tag) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_state128(unsigned long long* p, unsigned long long value, unsigned long long tag) {
  asm volatile("{\n.reg .b128 t;\nmov.b128 t, {%1, %2};\nst.relaxed.gpu.global.b128 [%0], t;\n}" ::"l"(p), "l"(value), "l"(tag)
               : "memory");
}
__device__ __forceinline__ unsigned ld_acq_sh(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_rel_sh(unsigned* p, unsigned v) {
  asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
// V = 2 doubles (one 128-bit access) or a multiple of 4 (256-bit accesses) with an L2 eviction-priority policy
template <int V> __device__ __forceinline__ void ldv_hint(double (&d)[V], const double* p, uint64_t policy) {
  uint32_t r[2 * V];
  if constexpr (V == 2) {
    ld_hint4(*reinterpret_cast<uint32_t(*)[4]>(r), p, policy);
  } else {
#pragma unroll
    for (int c = 0; c < V / 4; ++c)
      asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8], %9;"
                   : "=r"(r[8 * c]), "=r"(r[8 * c + 1]), "=r"(r[8 * c + 2]), "=r"(r[8 * c + 3]), "=r"(r[8 * c + 4]),
                     "=r"(r[8 * c + 5]), "=r"(r[8 * c + 6]), "=r"(r[8 * c + 7])
                   : "l"(p + 4 * c), "l"(policy)
                   : "memory");
  }
#pragma unroll
  for (int j = 0; j < V; ++j) d[j] = __hiloint2double(int(r[2 * j + 1]), int(r[2 * j]));
}
template <int V> __device__ __forceinline__ void stv_hint(double* p, const double (&d)[V], uint64_t policy) {
  uint32_t r[2 * V];
#pragma unroll
  for (int j = 0; j < V; ++j) {
    r[2 * j] = uint32_t(__double2loint(d[j]));
    r[2 * j + 1] = uint32_t(__double2hiint(d[j]));
  }
  if constexpr (V == 2) {
    st_hint4(p, *reinterpret_cast<const uint32_t(*)[4]>(r), policy);
  } else {
#pragma unroll
    for (int c = 0; c < V / 4; ++c)
      asm volatile("st.global.L1::no_allocate.L2::cache_hint.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8}, %9;" ::"l"(p + 4 * c),
                   "r"(r[8 * c]), "r"(r[8 * c + 1]), "r"(r[8 * c + 2]), "r"(r[8 * c + 3]), "r"(r[8 * c + 4]),
                   "r"(r[8 * c + 5]), "r"(r[8 * c + 6]), "r"(r[8 * c + 7]), "l"(policy)
                   : "memory");
  }
}

constexpr int L2_NW = 8, L2_D = 2, L2_S = 2, L2_KW = 10;   // the operating point of the i32 kernel
constexpr int L2_WT = L2_NW * 32;
// tile = 256 threads x V doubles x U
template <int U, int V = 2> struct L2Geom {
  static constexpr size_t TILE = size_t(L2_WT) * V * U;
  static constexpr size_t SMEM = L2_S * TILE * 8 + L2_S * 8 + 16;
};
constexpr size_t L2_TILE_MIN = L2Geom<4, 2>::TILE;  // the state array is sized for the smaller of the two tiles in use

template <int OP, int U, int MINB, int V>
__global__ void __launch_bounds__((L2_NW + 1) * 32, MINB)
scan_l2_f64_kernel(const double* in, double* out, size_t n, double init, int exclusive, unsigned long long* state,
                   unsigned long long launch_no, unsigned ntiles) {
  constexpr int NW = L2_NW, D = L2_D, S = L2_S, KW = L2_KW, WT = L2_WT, E = U * NW, Q = D + 2;
  constexpr size_t TILE = L2Geom<U, V>::TILE;
  constexpr unsigned FULL = 0xffffffffu;
  __shared__ double sm[2 * E + 1];
  __shared__ double red[2][NW];
  __shared__ double cq[Q];
  __shared__ unsigned cq_head, cq_tail;  // carries produced / consumed
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned long long G = gridDim.x;
  const double ident = didentity<OP>();
  if (threadIdx.x == 0) {
    cq_head = 0;
    cq_tail = 0;
  }
  __syncthreads();

  if (warp == NW) {  // ---------------- prefix warp ----------------
    double carry = exclusive ? init : ident;
    unsigned long long lo = 0;
    unsigned j = 0;
    for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += G, ++j) {
      double acc = ident;  // carry(tile) = carry(previous own tile) (+) aggregates of tiles [lo, tile), fixed grouping
      for (unsigned long long c0 = lo; c0 < tile; c0 += 32ull * KW) {
        bool pending = true;
        unsigned long long val[KW], tag[KW];
        while (pending) {
          pending = false;
#pragma unroll
          for (int k = 0; k < KW; ++k) {
            const unsigned long long idx = c0 + 32ull * k + lane;
            if (idx < tile) {
              ld_state128(state + 2 * idx, val[k], tag[k]);
            } else {
              val[k] = static_cast<unsigned long long>(__double_as_longlong(ident));
              tag[k] = launch_no;
            }
          }
#pragma unroll
          for (int k = 0; k < KW; ++k) pending |= tag[k] != launch_no;
          pending = __any_sync(FULL, pending);
        }
#pragma unroll
        for (int k = 0; k < KW; ++k) acc = dapply<OP>(0.0, acc, __longlong_as_double(static_cast<long long>(val[k])));
      }
      carry = dapply<OP>(0.0, carry, dwarp_reduce<OP>(acc));
      lo = tile;
      while (j - ld_acq_sh(&cq_tail) >= unsigned(Q)) {}  // queue full: wait for the workers
      if (lane == 0) {
        cq[j % Q] = carry;
        st_rel_sh(&cq_head, j + 1);
      }
      __syncwarp();
    }
    return;
  }

  // ---------------- worker warps ----------------
  constexpr unsigned TILE_BYTES = unsigned(TILE) * 8u;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* ring = reinterpret_cast<double*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + size_t(S) * TILE_BYTES);
  const uint64_t keep = l2_policy_evict_last(), stream = l2_policy_evict_first();
  auto bar_workers = [] { asm volatile("bar.sync 1, %0;" ::"n"(WT) : "memory"); };
  auto red_tile = [&](unsigned j) { return blockIdx.x + (unsigned long long)j * G; };
  auto issue = [&](unsigned j) {  // thread 0: arm stage j % S with reduce-tile j (whole tiles only)
    const unsigned long long t = red_tile(j);
    if (t < ntiles && (t + 1) * TILE <= n) {
      mbar_arrive_expect_tx(&full[j % S], TILE_BYTES);
      bulk_load_hint(ring + size_t(j % S) * TILE, in + size_t(t) * TILE, TILE_BYTES, &full[j % S], keep);
    }
  };
  if (threadIdx.x == 0) {
    for (int st = 0; st < S; ++st) mbar_init(&full[st], 1);
    mbar_fence_init();
    for (unsigned j = 0; j < unsigned(S); ++j) issue(j);
  }
  bar_workers();
  unsigned par = 0;
  auto reduce_tile = [&](unsigned j) {  // fold reduce-tile j, publish its aggregate, refill its stage
    const unsigned long long tile = red_tile(j);
    const size_t base = size_t(tile) * TILE;
    double a = ident;
    if (base + TILE <= n) {
      mbar_wait(&full[j % S], (j / S) & 1u);
      const double* stage = ring + size_t(j % S) * TILE;
#pragma unroll
      for (int k = 0; k < U * V / 2; ++k) {  // any fixed grouping serves for the aggregate: consecutive 16-byte reads
        const double2 q = *reinterpret_cast<const double2*>(stage + (k * WT + threadIdx.x) * 2);
        a = dapply<OP>(0.0, a, dapply<OP>(0.0, q.x, q.y));
      }
    } else {  // ragged last tile: guarded loads
      for (size_t i = base + threadIdx.x; i < n; i += WT) a = dapply<OP>(0.0, a, in[i]);
    }
    a = dwarp_reduce<OP>(a);
    if (lane == 0) red[par][warp] = a;
    bar_workers();  // every worker has read the stage
    if (warp == 0) {
      double v = lane < NW ? red[par][lane] : ident;
      v = dwarp_reduce<OP>(v);
      if (lane == 0) {
        st_state128(state + 2 * tile, static_cast<unsigned long long>(__double_as_longlong(v)), launch_no);
        issue(j + S);
      }
    }
    par ^= 1u;  // red[par] is rewritten two reduces later, with worker barriers in between
  };

  for (unsigned j = 0; j < unsigned(D); ++j) {  // prologue: run D tiles ahead
    if (red_tile(j) >= ntiles) break;
    reduce_tile(j);
  }
  unsigned it = 0;
  for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += G, ++it) {
    const size_t base = size_t(tile) * TILE;
    double x[U][V], lane_excl[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {  // second read of the tile: an L2 hit
      const size_t i0 = base + (size_t(u) * WT + threadIdx.x) * V;
      if (i0 + V <= n) {
        ldv_hint<V>(x[u], in + i0, stream);
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j) x[u][j] = i0 + j < n ? in[i0 + j] : ident;
      }
    }
    if (red_tile(it + D) < ntiles) reduce_tile(it + D);
#pragma unroll
    for (int u = 0; u < U; ++u) {  // local scan of the tile (registers)
#pragma unroll
      for (int j = 1; j < V; ++j) x[u][j] = dapply<OP>(0.0, x[u][j - 1], x[u][j]);
      double ws = x[u][V - 1];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const double y = __shfl_up_sync(FULL, ws, o);
        if (lane >= o) ws = dapply<OP>(0.0, y, ws);
      }
      const double ex = __shfl_up_sync(FULL, ws, 1);
      lane_excl[u] = lane == 0 ? ident : ex;
      if (lane == 31) sm[u * NW + warp] = ws;
    }
    bar_workers();
    if (warp == 0) {  // exclusive scan of the E = 64 (u, warp) totals, two per lane
      constexpr int EPL = (E + 31) / 32;
      double v[EPL];
      double run = ident;
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = lane * EPL + k;
        v[k] = e < E ? sm[e] : ident;
        run = dapply<OP>(0.0, run, v[k]);
      }
      double ws = run;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const double y = __shfl_up_sync(FULL, ws, o);
        if (lane >= o) ws = dapply<OP>(0.0, y, ws);
      }
      double ex = __shfl_up_sync(FULL, ws, 1);
      ex = lane == 0 ? ident : ex;
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = lane * EPL + k;
        if (e < E) sm[E + e] = ex;
        ex = dapply<OP>(0.0, ex, v[k]);
      }
    }
    while (ld_acq_sh(&cq_head) <= it) {}  // carry of this tile (normally long there)
    const double carry = cq[it % Q];
    bar_workers();
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const double p = dapply<OP>(0.0, dapply<OP>(0.0, carry, sm[E + u * NW + warp]), lane_excl[u]);
      double o[V];
#pragma unroll
      for (int j = 0; j < V; ++j) {
        if (exclusive) o[j] = j == 0 ? p : dapply<OP>(0.0, p, x[u][j - 1]);
        else o[j] = dapply<OP>(0.0, p, x[u][j]);
      }
      const size_t i0 = base + (size_t(u) * WT + threadIdx.x) * V;
      if (i0 + V <= n) {
        stv_hint<V>(out + i0, o, stream);
      } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
          if (i0 + j < n) out[i0 + j] = o[j];
      }
    }
    bar_workers();  // sm is reused; every worker has read its carry
    if (threadIdx.x == 0) st_rel_sh(&cq_tail, it + 1);
  }
}

template <int OP, int U, int MINB, int V>
cudaError_t scan_l2_f64(const Launch& L, Scratch& Sc, bool exclusive, double init, const double* in, double* out, size_t n) {
  constexpr size_t L2_TILE = L2Geom<U, V>::TILE, L2_SMEM = L2Geom<U, V>::SMEM;
  const size_t ntiles = (n + L2_TILE - 1) / L2_TILE;
  if (2 * ntiles > Sc.scan_state64_words || ntiles > 0x7fffffffu) return cudaErrorInvalidValue;
  auto kern = scan_l2_f64_kernel<OP, U, MINB, V>;
  static int ctas_per_sm = 0;
  if (ctas_per_sm == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L2_SMEM);
    if (e != cudaSuccess) return e;
    int per = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, (L2_NW + 1) * 32, L2_SMEM);
    if (e != cudaSuccess) return e;
    if (per < 1) return cudaErrorInvalidValue;
    ctas_per_sm = per;
  }
  size_t grid = size_t(L.sms) * ctas_per_sm;
  if (grid > ntiles) grid = ntiles;
  int excl = exclusive ? 1 : 0;
  unsigned long long launch_no = ++Sc.scan_launch64;  // starts at 1: the zero-initialised array holds no valid tag
  unsigned nt = (unsigned)ntiles;
  void* args[] = {&in, &out, &n, &init, &excl, &Sc.scan_state64, &launch_no, &nt};
  cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void*>(kern), dim3((unsigned)grid), dim3((L2_NW + 1) * 32), args,
                                              L2_SMEM, L.stream);
  ++*L.launches;
  return e;
}

size_t f64_chunk(size_t n) {  // elements per block of the chunked kernels: a multiple of 1024, at most MAX_PARTIALS chunks
  size_t chunk = 8192;
  const size_t need = (n + MAX_PARTIALS - 1) / MAX_PARTIALS;
  if (chunk < need) chunk = (need + 1023) / 1024 * 1024;
  return chunk;
}

template <int MAPF, bool HAS_IN1>
cudaError_t mr_op(const Launch& L, const Scratch& S, int red_op, double c, const double* in0, const double* in1, size_t n,
                  double* result) {
  const size_t chunk = f64_chunk(n);
  const unsigned grid = static_cast<unsigned>((n + chunk - 1) / chunk);
  double* partials = static_cast<double*>(S.partials);
  switch (red_op) {
    case FN_ADD: mapreduce_f64_kernel<MAPF, HAS_IN1, FN_ADD><<<grid, D_THREADS, 0, L.stream>>>(in0, in1, c, n, chunk, partials, S.ticket, result); break;
    case FN_MULT: mapreduce_f64_kernel<MAPF, HAS_IN1, FN_MULT><<<grid, D_THREADS, 0, L.stream>>>(in0, in1, c, n, chunk, partials, S.ticket, result); break;
    case FN_MAX: mapreduce_f64_kernel<MAPF, HAS_IN1, FN_MAX><<<grid, D_THREADS, 0, L.stream>>>(in0, in1, c, n, chunk, partials, S.ticket, result); break;
    default: return cudaErrorInvalidValue;
  }
  ++*L.launches;
  return cudaGetLastError();
}

template <int OP>
cudaError_t scan_op(const Launch& L, const Scratch& S, bool exclusive, double init, const double* in, double* out, size_t n) {
  const size_t chunk = f64_chunk(n);
  const unsigned grid = static_cast<unsigned>((n + chunk - 1) / chunk);
  double* partials = static_cast<double*>(S.partials);
  // phase 1: chunk totals (the Reduce kernel, one block per chunk, without its fold)
  mapreduce_f64_kernel<FN_IDENT, false, OP, false><<<grid, D_THREADS, 0, L.stream>>>(in, nullptr, 0.0, n, chunk, partials,
                                                                                   S.ticket, nullptr);
  const double start = exclusive ? init : (OP == FN_ADD ? 0.0 : (OP == FN_MULT ? 1.0 : -INFINITY));
  scan_f64_offsets_kernel<OP><<<1, D_THREADS, 0, L.stream>>>(partials, grid, start);
  if (exclusive) scan_f64_apply_kernel<OP, true><<<grid, D_THREADS, 0, L.stream>>>(in, out, n, chunk, partials);
  else scan_f64_apply_kernel<OP, false><<<grid, D_THREADS, 0, L.stream>>>(in, out, n, chunk, partials);
  *L.launches += 3;
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_map_f64(const Launch& L, int fn, bool has_in1, double c, const double* in0, const double* in1,
                           const double* in2, double* out, size_t n) {
  if (n == 0) return cudaSuccess;
  const size_t tile = size_t(D_THREADS) * 4 * 2;
  const size_t grid = (n + tile - 1) / tile;
  if (grid > 0x7fffffffu) return cudaErrorInvalidValue;
#define SKEL_F64_MAP(FN, NIN) map_f64_kernel<FN, NIN><<<(unsigned)grid, D_THREADS, 0, L.stream>>>(c, in0, in1, in2, out, n)
  if (in2) SKEL_F64_MAP(FN_ADD, 3);
  else if (has_in1) {
    switch (fn) {
      case FN_ADD: SKEL_F64_MAP(FN_ADD, 2); break;
      case FN_MULT: SKEL_F64_MAP(FN_MULT, 2); break;
      case FN_MAX: SKEL_F64_MAP(FN_MAX, 2); break;
      case FN_SAXPY: SKEL_F64_MAP(FN_SAXPY, 2); break;
      default: return cudaErrorInvalidValue;
    }
  } else {
    switch (fn) {
      case FN_ADD: SKEL_F64_MAP(FN_ADD, 1); break;
      case FN_MULT: SKEL_F64_MAP(FN_MULT, 1); break;
      case FN_MAX: SKEL_F64_MAP(FN_MAX, 1); break;
      default: return cudaErrorInvalidValue;
    }
  }
#undef SKEL_F64_MAP
  ++*L.launches;
  return cudaGetLastError();
}

cudaError_t launch_mapreduce_f64(const Launch& L, const Scratch& S, int map_fn, bool has_in1, int red_op, double c,
                                 const double* in0, const double* in1, size_t n, double* result) {
  switch (map_fn) {
    case FN_IDENT: return mr_op<FN_IDENT, false>(L, S, red_op, c, in0, in1, n, result);
    case FN_ADD: return has_in1 ? mr_op<FN_ADD, true>(L, S, red_op, c, in0, in1, n, result) : mr_op<FN_ADD, false>(L, S, red_op, c, in0, in1, n, result);
    case FN_MULT: return has_in1 ? mr_op<FN_MULT, true>(L, S, red_op, c, in0, in1, n, result) : mr_op<FN_MULT, false>(L, S, red_op, c, in0, in1, n, result);
    case FN_MAX: return has_in1 ? mr_op<FN_MAX, true>(L, S, red_op, c, in0, in1, n, result) : mr_op<FN_MAX, false>(L, S, red_op, c, in0, in1, n, result);
    case FN_SAXPY: return mr_op<FN_SAXPY, true>(L, S, red_op, c, in0, in1, n, result);
  }
  return cudaErrorInvalidValue;
}

size_t scan_f64_state_words(size_t n) { return n >= SCAN_F64_L2_MIN ? 2 * ((n + L2_TILE_MIN - 1) / L2_TILE_MIN) : 0; }

// A thread owns V = 8 contiguous doubles per step (two 256-bit accesses), U = 2 steps per 32 KB tile: the cross-lane
// scans (10 shuffles of 64-bit values + 5 dependent DADDs each) are what limits the fp64 form, and their number per
// byte falls with V. Measured at 2^25 (16 B/elem): V = 2, U = 4: 133 us; V = 4, U = 2: 116 us; V = 8, U = 1 (16 KB tiles,
// 3 CTAs per SM): 112 us; V = 16, U = 1: 113 us; V = 8, U = 2: 103 us. Operands that are only 16-byte aligned (adopted
// pointers) take V = 2.
template <int OP>
cudaError_t scan_l2_f64_any(const Launch& L, Scratch& S, bool exclusive, double init, const double* in, double* out, size_t n) {
  if (reinterpret_cast<uintptr_t>(in) % 32 == 0 && reinterpret_cast<uintptr_t>(out) % 32 == 0)
    return scan_l2_f64<OP, 2, 2, 8>(L, S, exclusive, init, in, out, n);
  return scan_l2_f64<OP, 4, 3, 2>(L, S, exclusive, init, in, out, n);
}

cudaError_t launch_scan_f64(const Launch& L, Scratch& S, int op, bool exclusive, double init, const double* in,
                            double* out, size_t n) {
  if (n == 0) return cudaSuccess;
  if (n >= SCAN_F64_L2_MIN && reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0) {
    switch (op) {
      case FN_ADD: return scan_l2_f64_any<FN_ADD>(L, S, exclusive, init, in, out, n);
      case FN_MULT: return scan_l2_f64_any<FN_MULT>(L, S, exclusive, init, in, out, n);
      case FN_MAX: return scan_l2_f64_any<FN_MAX>(L, S, exclusive, init, in, out, n);
    }
    return cudaErrorInvalidValue;
  }
  switch (op) {
    case FN_ADD: return scan_op<FN_ADD>(L, S, exclusive, init, in, out, n);
    case FN_MULT: return scan_op<FN_MULT>(L, S, exclusive, init, in, out, n);
    case FN_MAX: return scan_op<FN_MAX>(L, S, exclusive, init, in, out, n);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_overlap1d_f64(const Launch& L, const Weights1D64& w, int r, int edge, double pad, int axis,
                                 const double* in, double* out, size_t rows, size_t cols) {
  const size_t total = rows * ((cols + 3) / 4);  // a thread owns 4 consecutive elements of a row
  if (rows * cols == 0) return cudaSuccess;
  size_t grid = (total + D_THREADS - 1) / D_THREADS;
  const size_t cap = size_t(L.sms) * 64;
  if (grid > cap) grid = cap;
  const bool rows_fast = axis == 0 && r >= 0 && r <= 16 && cols % 4 == 0 && cols >= 64 &&
                         reinterpret_cast<uintptr_t>(in) % 32 == 0 && reinterpret_cast<uintptr_t>(out) % 32 == 0;
  if (rows_fast) {
    const int R = r <= 4 ? 4 : (r <= 8 ? 8 : 16);
    Weights1D64 wp;
    for (double& x : wp.w) x = 0.0;
    for (int k = 0; k <= 2 * r; ++k) wp.w[k + R - r] = w.w[k];
    if (R == 4) overlap1d_f64_rows_kernel<4><<<(unsigned)grid, D_THREADS, 0, L.stream>>>(wp, r, edge, pad, in, out, rows, cols);
    else if (R == 8) overlap1d_f64_rows_kernel<8><<<(unsigned)grid, D_THREADS, 0, L.stream>>>(wp, r, edge, pad, in, out, rows, cols);
    else overlap1d_f64_rows_kernel<16><<<(unsigned)grid, D_THREADS, 0, L.stream>>>(wp, r, edge, pad, in, out, rows, cols);
  } else {
    overlap1d_f64_kernel<<<(unsigned)grid, D_THREADS, 0, L.stream>>>(w, r, edge, pad, axis, in, out, rows, cols);
  }
  ++*L.launches;
  return cudaGetLastError();
}

cudaError_t launch_overlap2d_f64(const Launch& L, const Weights2D64& w, int ry, int rx, int edge, double pad,
                                 const double* in, double* out, size_t rows, size_t cols) {
  const size_t total = rows * cols;
  if (total == 0) return cudaSuccess;
  size_t grid = (total + D_THREADS - 1) / D_THREADS;
  const size_t cap = size_t(L.sms) * 64;
  if (grid > cap) grid = cap;
  overlap2d_f64_kernel<<<(unsigned)grid, D_THREADS, 0, L.stream>>>(w, ry, rx, edge, pad, in, out, rows, cols);
  ++*L.launches;
  return cudaGetLastError();
}

}  // namespace skel
