// Host-side launch interface of the skeleton kernels (internal to libskel.so).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace skel {

enum : int { DT_F32 = 0, DT_I32 = 1, DT_F64 = 2 };

struct Launch {
  cudaStream_t stream;
  int sms;            // SM count of the device (148 on B200)
  int* launches;      // incremented once per kernel launch
  // dynamic tile assignment of the persistent TMA kernels: a device counter that is never reset, and the host's copy
  // of the value it will have when the next launch starts (launches of a context are ordered on one stream)
  unsigned* tile_ctr;
  unsigned* tile_next;
};

struct Scratch {       // device scratch owned by the context (see api.cu)
  void* partials;      // >= MAX_PARTIALS 8-byte slots (reduce partials, scan block sums)
  unsigned* ticket;    // reduce: atomicInc ticket (self-resetting); +2: packed word of the iatom end; +4: start-order ticket of the tagged end
  unsigned long long* red_tagged = nullptr;  // reduce, "*_tag" variants: MAX_PARTIALS + 8 (partial bits, launch number) slots (per block, then the 8 second-level ones), zero-initialised
  mutable uint32_t red_epoch = 0;            // launch number of the last tagged Reduce (host side)
  unsigned* scan_ticket;        // scan: dynamic tile id counter (reset by the last tile)
  unsigned long long* scan_state;  // scan: per-tile (epoch|status|value) words, zero-initialised
  size_t scan_state_tiles;      // capacity of scan_state in tiles
  uint32_t scan_epoch;          // incremented per look-back launch (host side)
  unsigned long long* scan_state64 = nullptr;  // fp64 single-pass scan: 16 bytes per tile (aggregate, launch number)
  size_t scan_state64_words = 0;               // capacity in 8-byte words, zero-initialised, never cleared
  unsigned long long scan_launch64 = 0;        // launch number of the last fp64 single-pass scan (tags the states)
};
constexpr int MAX_PARTIALS = 8192;

// ---- Map -------------------------------------------------------------------------------------
int map_variant_count();
const char* map_variant_name(int v);
// whether variant v can run this call (alignment / size constraints)
bool map_variant_ok(int v, const void* in0, const void* in1, const void* out, size_t n);
cudaError_t launch_map(const Launch& L, int v, int dtype, int fn, bool has_in1, uint32_t cbits,
                       const void* in0, const void* in1, void* out, size_t n);

// three-vector Map, MULADD: out[i] = in0[i] * in1[i] + in2[i] (same variant table; alignment of all four pointers)
cudaError_t launch_map3(const Launch& L, int v, int dtype, const void* in0, const void* in1, const void* in2, void* out,
                        size_t n);

// ---- Reduce / MapReduce (map_fn = FN_IDENT for plain Reduce) --------------------------------------
int reduce_variant_count();
const char* reduce_variant_name(int v);
bool reduce_variant_ok(int v, const void* in0, const void* in1, size_t n);
cudaError_t launch_mapreduce(const Launch& L, const Scratch& S, int v, int dtype, int map_fn, bool has_in1,
                             int red_op, uint32_t cbits, const void* in0, const void* in1, size_t n,
                             void* result /* device, one element */,
                             bool reverse = false /* chunk variants: walk the operands from the end to the front (same
                                                     result bits; api.cu uses it to meet what the previous launch left in L2) */);

// ---- row-wise Reduce on a matrix: out[i] = in[i][0] (+) ... (+) in[i][cols-1] (reduce.cu) ----------------
int reduce_rows_variant_count();
const char* reduce_rows_variant_name(int v);
bool reduce_rows_variant_ok(int v, const void* in, size_t rows, size_t cols);
cudaError_t launch_reduce_rows(const Launch& L, int v, int dtype, int op, const void* in, size_t rows, size_t cols,
                               void* out /* device, rows elements */);

// ---- Scan ------------------------------------------------------------------------------------
int scan_variant_count();
const char* scan_variant_name(int v);
bool scan_variant_ok(int v, int dtype, const void* in, const void* out, size_t n);
cudaError_t launch_scan(const Launch& L, Scratch& S, int v, int dtype, int op, bool exclusive, uint32_t init_bits,
                        const void* in, void* out, size_t n);
size_t scan_tiles_needed(size_t n);

// ---- MapOverlap ---------------------------------------------------------------------------------
// Weights travel as 32-bit images typed float: for int32 elements (dtype = DT_I32) w[] holds the int32 bit patterns
// and so does `pad`; the data pointers are typed float* for the same reason (common.cuh StencilOps).
struct Weights1D { float w[129]; };   // 2r+1 <= 129 taps, passed by value (constant bank)
struct Weights2D { float w[17 * 17]; };

// Radii the tiled kernels are instantiated for: {1, 2, 3, 4, 8, 16} in 1D, square {1..4} in 2D, {1, 2, 3, 4, 8} for the
// fused separable pair. Any other radius up to the largest runs the NEXT instantiated one with the weights zero-padded
// at both ends (a radius-5 filter IS a radius-8 filter whose outer taps are 0): every tap keeps its place in the
// ascending order, the extra fused multiply-adds add 0 * x~ = 0, so for finite data the result has the same bits
// (a non-finite x~ within the padded reach of an output, but outside its real reach, would turn it into NaN: the
// direct variant is the one to force for such data).
inline int padded_radius_1d(int r) { return r <= 4 ? (r < 1 ? 1 : r) : (r <= 8 ? 8 : (r <= 16 ? 16 : -1)); }
inline Weights1D pad_weights_1d(const Weights1D& w, int r, int R) {
  Weights1D o;
  for (float& x : o.w) x = 0.f;
  for (int k = 0; k <= 2 * r; ++k) o.w[k + (R - r)] = w.w[k];
  return o;
}
inline Weights2D pad_weights_2d(const Weights2D& w, int ry, int rx, int R) {  // (2ry+1) x (2rx+1) -> (2R+1)^2
  Weights2D o;
  for (float& x : o.w) x = 0.f;
  for (int a = 0; a <= 2 * ry; ++a)
    for (int b = 0; b <= 2 * rx; ++b) o.w[(a + R - ry) * (2 * R + 1) + (b + R - rx)] = w.w[a * (2 * rx + 1) + b];
  return o;
}

int overlap1d_variant_count();
const char* overlap1d_variant_name(int v);
bool overlap1d_variant_ok(int v, int dtype, int r, const void* in, const void* out, size_t rows, size_t cols);
// vector: rows = 1. Row-wise on a matrix: every row independently.
cudaError_t launch_overlap1d_rows(const Launch& L, int v, int dtype, const Weights1D& w, int r, int edge, float pad,
                                  const float* in, float* out, size_t rows, size_t cols);

int overlap1d_col_variant_count();
const char* overlap1d_col_variant_name(int v);
bool overlap1d_col_variant_ok(int v, int dtype, int r, const void* in, const void* out, size_t rows, size_t cols);
cudaError_t launch_overlap1d_cols(const Launch& L, int v, int dtype, const Weights1D& w, int r, int edge, float pad,
                                  const float* in, float* out, size_t rows, size_t cols);

int overlap2d_variant_count();
const char* overlap2d_variant_name(int v);
bool overlap2d_variant_ok(int v, int dtype, int ry, int rx, const void* in, const void* out, size_t rows, size_t cols);
cudaError_t launch_overlap2d(const Launch& L, int v, int dtype, const Weights2D& w, int ry, int rx, int edge, float pad,
                             const float* in, float* out, size_t rows, size_t cols);

// ---- fused chain [Map(f, c)] -> MapOverlap1D -> [Reduce(op)] on one f32 vector (fused.cu) -----------
// map_fn = FN_IDENT (100): no Map in the chain (map_out unused); red_op = FUSED_NO_REDUCE: no Reduce.
constexpr int FUSED_NO_REDUCE = -1;
bool fused_chain_ok(int map_fn, int r, int red_op, const void* in, const void* map_out, const void* ov_out, size_t n);
cudaError_t launch_fused_chain(const Launch& L, const Scratch& S, int map_fn, uint32_t cbits, const Weights1D& w, int r,
                               int edge, float pad, int red_op, const float* in, float* map_out, float* ov_out, size_t n,
                               float* result /* device, one element; unused without a Reduce */);

// ---- fused separable MapOverlap on a matrix (separable.cu); variant 0 = two 1D passes (api.cu) -------
int separable_variant_count();
const char* separable_variant_name(int v);
bool separable_variant_ok(int v, int r_row, int r_col, const void* in, const void* out, size_t rows, size_t cols);
cudaError_t launch_separable_fused(const Launch& L, int v, const Weights1D& wrow, const Weights1D& wcol, int r_row,
                                   int r_col, int edge, float pad, const float* in, float* out, size_t rows, size_t cols);

// ---- fp64 elements (f64.cu; dtype = DT_F64): one kernel per skeleton, no variant table ---------------------------
struct Weights1D64 { double w[129]; };
struct Weights2D64 { double w[17 * 17]; };
// in2 != NULL: three-vector MULADD (fn ignored); else out = f(in0, in1 or c)
cudaError_t launch_map_f64(const Launch& L, int fn, bool has_in1, double c, const double* in0, const double* in1,
                           const double* in2, double* out, size_t n);
cudaError_t launch_mapreduce_f64(const Launch& L, const Scratch& S, int map_fn, bool has_in1, int red_op, double c,
                                 const double* in0, const double* in1, size_t n, double* result /* device */);
// n >= SCAN_F64_L2_MIN (16-byte aligned operands): single pass ("l2ahead"), needs scan_f64_state_words(n) words of
// Scratch::scan_state64; smaller n: three kernels.
constexpr size_t SCAN_F64_L2_MIN = size_t(1) << 20;
size_t scan_f64_state_words(size_t n);
cudaError_t launch_scan_f64(const Launch& L, Scratch& S, int op, bool exclusive, double init, const double* in,
                            double* out, size_t n);
// axis 0: along the rows (a vector is rows = 1), 1: along the columns
cudaError_t launch_overlap1d_f64(const Launch& L, const Weights1D64& w, int r, int edge, double pad, int axis,
                                 const double* in, double* out, size_t rows, size_t cols);
cudaError_t launch_overlap2d_f64(const Launch& L, const Weights2D64& w, int ry, int rx, int edge, double pad,
                                 const double* in, double* out, size_t rows, size_t cols);

// ---- FP32 FMA roofline probe (probe.cu) ------------------------------------------------------------
cudaError_t launch_fma_probe(const Launch& L, float* scratch /* device, >= 1 float */, double* fma_count);
// FFMA2 stream with nl in {0, 1, 2, 4, 8} LDS.128 per 144 FMA-pipe cycles; in64: device, 64 floats
cudaError_t launch_fma_lds_probe(const Launch& L, int nl, const float* in64, float* scratch, double* fma_count);

// tiled variants (v >= 1) of one radius; specialised in overlap2d_inst.cu, one translation unit per radius
template <int R>
cudaError_t launch_overlap2d_tiled(const Launch& L, int v, int dtype, const Weights2D& w, int edge, float pad,
                                   const float* in, float* out, size_t rows, size_t cols);
template <int R>
cudaError_t launch_overlap1d_cols_tiled(const Launch& L, int v, int dtype, const Weights1D& w, int edge, float pad,
                                        const float* in, float* out, size_t rows, size_t cols);

}  // namespace skel
