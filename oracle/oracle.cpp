// CPU ORACLE — TEST INFRASTRUCTURE ONLY. Not part of the product path.
//
// Plain, slow, obviously-correct definitions of the SkePU-style data-parallel skeletons that
// arxiv 1405.2915 names ("map, mapoverlap, scan, reduce, ...", §III; "map, farm,
// scan and reduce") applied to the payload of Vector/Matrix containers (PAPER.md
// L111). The paper names the skeletons but prints no formula; every definition below is the
// textbook higher-order function, with the readings listed in DESIGN.md §"Readings" (taken from
// SURVEY.md §8(c).1-(c).6). Each function cites the reading it follows.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library. It shares no code, header, table or constant with paper_1405_2915_b200/csrc
// or include/skel.h: the enum values below are restated, not included.
//
// Arithmetic: fp32 inputs are widened to double and everything is computed in fp64 in the order
// the definition states (sums of Reduce/MapReduce use Neumaier compensation so that the oracle's own
// error, ~1e-16 * sum|t|, is irrelevant next to the 1e-5 / 2e-6 tolerances). int32 paths use
// two's-complement wrap-around (mod 2^32) arithmetic on uint32_t (reading (c).2 ii).
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): closed forms (sum i = n(n-1)/2, scan of
// ones = indices, stencil of a constant = constant * sum w, constant-0 border closed form,
// cyclic stencil == circular correlation computed with numpy roll / FFT-free definition),
// impulse / one-hot-weight shift tests (orientation, indexing, edge policy, bit-exact), split and
// permutation invariants, the separable identity (row pass . col pass == dense outer-product
// filter), transpose symmetry, library special cases (numpy cumsum / correlate / math.fsum), and
// brute-force pure-Python loops on tiny inputs; the int32 MapOverlap functions against exact Python integers,
// numpy.correlate on int64, one-hot shifts and the fp64 functions above on small values (where both are exact).
// The fp64-element functions (binary128 arithmetic) against exact rationals (Python Fraction), cancellation cases a
// plain fp64 loop gets wrong, and the fp32-element functions on fp32-representable data.
// No function here is "parity unpinned".
//
// The `#pragma omp parallel for` lines only take effect in the -fopenmp build (liboracle_omp.so),
// which runs the SAME loops over independent outputs in parallel; it is used for timing and for
// full-size parity runs. Reduce and Scan are sequential in both builds.

#include <cmath>
#include <cstddef>
#include <cstdint>

namespace {

// restated ABI values (see header comment): user functions, edge policies, scan modes, axes
enum { FN_ADD = 0, FN_MULT = 1, FN_MAX = 2, FN_SAXPY = 3 };
enum { EDGE_CONSTANT = 0, EDGE_DUPLICATE = 1, EDGE_CYCLIC = 2 };
enum { SCAN_INCLUSIVE = 0, SCAN_EXCLUSIVE = 1 };
enum { AXIS_ROW = 0, AXIS_COL = 1 };

inline uint32_t u32(int32_t v) { return static_cast<uint32_t>(v); }
inline int32_t i32(uint32_t v) { return static_cast<int32_t>(v); }

// reading (c).1: add a+b, mult a*b, max (a<b ? b : a), saxpy c*a+b; fp64
inline double f_apply(int fn, double c, double a, double b) {
  switch (fn) {
    case FN_ADD: return a + b;
    case FN_MULT: return a * b;
    case FN_MAX: return a < b ? b : a;
    case FN_SAXPY: return c * a + b;
  }
  return NAN;
}

// int32, wrap mod 2^32 (reading (c).2 ii, (c).3 iii)
inline int32_t i_apply(int fn, int32_t c, int32_t a, int32_t b) {
  switch (fn) {
    case FN_ADD: return i32(u32(a) + u32(b));
    case FN_MULT: return i32(u32(a) * u32(b));
    case FN_MAX: return a < b ? b : a;
    case FN_SAXPY: return i32(u32(c) * u32(a) + u32(b));
  }
  return 0;
}

// Neumaier-compensated running sum
struct NSum {
  double s = 0.0, comp = 0.0;
  void add(double v) {
    double t = s + v;
    if (std::fabs(s) >= std::fabs(v)) comp += (s - t) + v; else comp += (v - t) + s;
    s = t;
  }
  double value() const { return s + comp; }
};

inline ptrdiff_t clampi(ptrdiff_t j, ptrdiff_t lo, ptrdiff_t hi) { return j < lo ? lo : (j > hi ? hi : j); }
// CYCLIC (reading 19): the index wraps around, x~[j] = x[j mod n] with the
// mathematical (non-negative) remainder; in 2D each index wraps on its own.
inline ptrdiff_t wrapi(ptrdiff_t j, ptrdiff_t n) { ptrdiff_t m = j % n; return m < 0 ? m + n : m; }

// reading (c).5: x~[j] = x[j] inside; CONSTANT -> pad; DUPLICATE -> x[clamp(j,0,n-1)].
// `stride` lets the same definition walk a matrix column.
template <typename T>
inline double ext1(const T* x, ptrdiff_t n, ptrdiff_t stride, ptrdiff_t j, int edge, double pad) {
  if (j >= 0 && j < n) return static_cast<double>(x[j * stride]);
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) return static_cast<double>(x[wrapi(j, n) * stride]);
  return static_cast<double>(x[clampi(j, 0, n - 1) * stride]);
}

// one output of MapOverlap 1D: sum_{k=-r..r} w[k+r] * x~[i+k], increasing k (correlation, no flip)
template <typename T>
inline void overlap1_at(const float* w, int r, int edge, double pad, const T* x, ptrdiff_t n,
                        ptrdiff_t stride, ptrdiff_t i, double* out, double* absout) {
  double acc = 0.0, aacc = 0.0;
  for (int k = -r; k <= r; ++k) {
    double t = static_cast<double>(w[k + r]) * ext1(x, n, stride, i + k, edge, pad);
    acc += t;
    aacc += std::fabs(t);
  }
  *out = acc;
  if (absout) *absout = aacc;
}

template <typename T>
void overlap1_matrix(const float* w, int r, int edge, double pad, int axis, const T* X,
                     ptrdiff_t rows, ptrdiff_t cols, double* out, double* absout) {
  // row-wise: every row is an independent vector of length cols; col-wise: every column is an
  // independent vector of length rows (reading (c).5).
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < rows; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j) {
      double* a = absout ? absout + i * cols + j : nullptr;
      if (axis == AXIS_ROW)
        overlap1_at(w, r, edge, pad, X + i * cols, cols, 1, j, out + i * cols + j, a);
      else
        overlap1_at(w, r, edge, pad, X + j, rows, cols, i, out + i * cols + j, a);
    }
}

// reading (c).6: X~[p][q] with each index clamped independently (DUPLICATE) or pad (CONSTANT)
template <typename T>
inline double ext2(const T* X, ptrdiff_t rows, ptrdiff_t cols, ptrdiff_t p, ptrdiff_t q, int edge,
                   double pad) {
  if (p >= 0 && p < rows && q >= 0 && q < cols) return static_cast<double>(X[p * cols + q]);
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) return static_cast<double>(X[wrapi(p, rows) * cols + wrapi(q, cols)]);
  return static_cast<double>(X[clampi(p, 0, rows - 1) * cols + clampi(q, 0, cols - 1)]);
}

template <typename T>
void overlap2_rows(const float* W, int ry, int rx, int edge, double pad, const T* X, ptrdiff_t rows,
                   ptrdiff_t cols, ptrdiff_t row0, ptrdiff_t row1, double* out, double* absout) {
  const int fw = 2 * rx + 1;
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = row0; i < row1; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j) {
      double acc = 0.0, aacc = 0.0;
      for (int a = -ry; a <= ry; ++a)      // a outer
        for (int b = -rx; b <= rx; ++b) {  // b inner
          double t = static_cast<double>(W[(a + ry) * fw + (b + rx)]) *
                     ext2(X, rows, cols, i + a, j + b, edge, pad);
          acc += t;
          aacc += std::fabs(t);
        }
      out[(i - row0) * cols + j] = acc;
      if (absout) absout[(i - row0) * cols + j] = aacc;
    }
}

// ---- int32 MapOverlap ("i32 element types for all skeletons"; reading 26): the same
// definitions with int32 data, int32 weights and an int32 pad value; every product and every sum wraps modulo 2^32
// (computed on uint32_t, like the int32 Map / Reduce / Scan: reading (c).2 ii). x~ follows the same edge policies.
inline uint32_t iext1(const int32_t* x, ptrdiff_t n, ptrdiff_t stride, ptrdiff_t j, int edge, int32_t pad) {
  if (j >= 0 && j < n) return u32(x[j * stride]);
  if (edge == EDGE_CONSTANT) return u32(pad);
  if (edge == EDGE_CYCLIC) return u32(x[wrapi(j, n) * stride]);
  return u32(x[clampi(j, 0, n - 1) * stride]);
}

inline int32_t ioverlap1_at(const int32_t* w, int r, int edge, int32_t pad, const int32_t* x, ptrdiff_t n,
                            ptrdiff_t stride, ptrdiff_t i) {
  uint32_t acc = 0;
  for (int k = -r; k <= r; ++k) acc += u32(w[k + r]) * iext1(x, n, stride, i + k, edge, pad);
  return i32(acc);
}

inline uint32_t iext2(const int32_t* X, ptrdiff_t rows, ptrdiff_t cols, ptrdiff_t p, ptrdiff_t q, int edge, int32_t pad) {
  if (p >= 0 && p < rows && q >= 0 && q < cols) return u32(X[p * cols + q]);
  if (edge == EDGE_CONSTANT) return u32(pad);
  if (edge == EDGE_CYCLIC) return u32(X[wrapi(p, rows) * cols + wrapi(q, cols)]);
  return u32(X[clampi(p, 0, rows - 1) * cols + clampi(q, 0, cols - 1)]);
}

// ---- fp64 elements (SURVEY.md 8(f) f2 "f64 element types for all skeletons"; reading 27) ------------------
// The oracle of an fp64 path cannot be fp64: it computes in binary128 (__float128, 113-bit significand; plain
// arithmetic only, no libquadmath call). The product of two fp64 values (106 bits) is EXACT in binary128, sums carry
// ~1e-34 relative error per step, and the result is rounded to fp64 once at the end. Pinned against exact rational
// arithmetic (Python Fraction) in tests/test_oracle_pins.py.
typedef __float128 q128;
inline q128 q_apply(int fn, q128 c, q128 a, q128 b) {
  switch (fn) {
    case FN_ADD: return a + b;
    case FN_MULT: return a * b;
    case FN_MAX: return a < b ? b : a;
    case FN_SAXPY: return c * a + b;
  }
  return 0;
}
inline q128 q_abs(q128 v) { return v < 0 ? -v : v; }

inline q128 qext1(const double* x, ptrdiff_t n, ptrdiff_t stride, ptrdiff_t j, int edge, double pad) {
  if (j >= 0 && j < n) return x[j * stride];
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) return x[wrapi(j, n) * stride];
  return x[clampi(j, 0, n - 1) * stride];
}
inline void qoverlap1_at(const double* w, int r, int edge, double pad, const double* x, ptrdiff_t n, ptrdiff_t stride,
                         ptrdiff_t i, double* out, double* absout) {
  q128 acc = 0, aacc = 0;
  for (int k = -r; k <= r; ++k) {
    const q128 t = q128(w[k + r]) * qext1(x, n, stride, i + k, edge, pad);  // exact
    acc += t;
    aacc += q_abs(t);
  }
  *out = static_cast<double>(acc);
  if (absout) *absout = static_cast<double>(aacc);
}
inline q128 qext2(const double* X, ptrdiff_t rows, ptrdiff_t cols, ptrdiff_t p, ptrdiff_t q, int edge, double pad) {
  if (p >= 0 && p < rows && q >= 0 && q < cols) return X[p * cols + q];
  if (edge == EDGE_CONSTANT) return pad;
  if (edge == EDGE_CYCLIC) return X[wrapi(p, rows) * cols + wrapi(q, cols)];
  return X[clampi(p, 0, rows - 1) * cols + clampi(q, 0, cols - 1)];
}

}  // namespace

extern "C" {

int oracle_abi_version(void) { return 3; }

// ---- Map (reading (c).1). out[i] = f(in0[i], b_i), b_i = in1[i] or the constant c (rounded to
// fp32 first, reading (c).1 iii). Result in fp64.
void oracle_map_f32(int fn, double c, const float* in0, const float* in1, size_t n, double* out) {
  const double c32 = static_cast<double>(static_cast<float>(c));
  const ptrdiff_t N = static_cast<ptrdiff_t>(n);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < N; ++i) {
    double a = in0[i];
    double b = in1 ? static_cast<double>(in1[i]) : c32;
    out[i] = f_apply(fn, c32, a, b);
  }
}

// ---- three-vector Map: MULADD out[i] = in0[i] * in1[i] + in2[i]; fp64 (the product of two
// fp32 values is exact in fp64), int32 wraps.
void oracle_map3_f32(const float* in0, const float* in1, const float* in2, size_t n, double* out) {
  const ptrdiff_t N = static_cast<ptrdiff_t>(n);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < N; ++i)
    out[i] = static_cast<double>(in0[i]) * static_cast<double>(in1[i]) + static_cast<double>(in2[i]);
}

void oracle_map3_i32(const int32_t* in0, const int32_t* in1, const int32_t* in2, size_t n, int32_t* out) {
  for (size_t i = 0; i < n; ++i) out[i] = i32(u32(in0[i]) * u32(in1[i]) + u32(in2[i]));
}

void oracle_map_i32(int fn, int32_t c, const int32_t* in0, const int32_t* in1, size_t n, int32_t* out) {
  for (size_t i = 0; i < n; ++i) out[i] = i_apply(fn, c, in0[i], in1 ? in1[i] : c);
}

// ---- Reduce (reading (c).2). acc = in[0]; acc = acc (+) in[i]. n == 0 -> returns -1.
// abs_sum receives sum |in[i]| (the tolerance denominator of BASELINE.json L5).
int oracle_reduce_f32(int op, const float* in, size_t n, double* result, double* abs_sum) {
  if (n == 0) return -1;
  NSum s, as;
  double acc = in[0];
  s.add(acc);
  as.add(std::fabs(acc));
  for (size_t i = 1; i < n; ++i) {
    double v = in[i];
    if (op == FN_ADD) s.add(v); else acc = f_apply(op, 0.0, acc, v);
    as.add(std::fabs(v));
  }
  *result = (op == FN_ADD) ? s.value() : acc;
  if (abs_sum) *abs_sum = as.value();
  return 0;
}

// ---- row-wise Reduce on a matrix: out[i] = Reduce(row i), every row on its own,
// by the vector Reduce above (that IS the definition). cols == 0 -> returns -1.
int oracle_reduce_rows_f32(int op, const float* in, size_t rows, size_t cols, double* result, double* abs_sum) {
  if (cols == 0) return -1;
#pragma omp parallel for schedule(static)
  for (long long i = 0; i < (long long)rows; ++i)
    oracle_reduce_f32(op, in + size_t(i) * cols, cols, result + i, abs_sum ? abs_sum + i : nullptr);
  return 0;
}

int oracle_reduce_i32(int op, const int32_t* in, size_t n, int32_t* result, int64_t* exact_i64);
int oracle_reduce_rows_i32(int op, const int32_t* in, size_t rows, size_t cols, int32_t* result) {
  if (cols == 0) return -1;
#pragma omp parallel for schedule(static)
  for (long long i = 0; i < (long long)rows; ++i) {
    int64_t ex;
    oracle_reduce_i32(op, in + size_t(i) * cols, cols, result + i, &ex);
  }
  return 0;
}

// exact_i64 receives the un-wrapped int64 sum for op == add (information only).
int oracle_reduce_i32(int op, const int32_t* in, size_t n, int32_t* result, int64_t* exact_i64) {
  if (n == 0) return -1;
  int32_t acc = in[0];
  int64_t ex = in[0];
  for (size_t i = 1; i < n; ++i) {
    acc = i_apply(op, 0, acc, in[i]);
    ex += in[i];
  }
  *result = acc;
  if (exact_i64) *exact_i64 = ex;
  return 0;
}

// ---- MapReduce (reading (c).3). acc = f(in0[0], b_0); acc = acc (+) f(in0[i], b_i); the mapped
// vector is never stored. abs_sum = sum |f(...)|.
int oracle_mapreduce_f32(int map_f, int red_op, double c, const float* in0, const float* in1,
                         size_t n, double* result, double* abs_sum) {
  if (n == 0) return -1;
  const double c32 = static_cast<double>(static_cast<float>(c));
  NSum s, as;
  double acc = 0.0;
  for (size_t i = 0; i < n; ++i) {
    double t = f_apply(map_f, c32, in0[i], in1 ? static_cast<double>(in1[i]) : c32);
    if (i == 0) { acc = t; s.add(t); }
    else if (red_op == FN_ADD) s.add(t);
    else acc = f_apply(red_op, 0.0, acc, t);
    as.add(std::fabs(t));
  }
  *result = (red_op == FN_ADD) ? s.value() : acc;
  if (abs_sum) *abs_sum = as.value();
  return 0;
}

int oracle_mapreduce_i32(int map_f, int red_op, int32_t c, const int32_t* in0, const int32_t* in1,
                         size_t n, int32_t* result) {
  if (n == 0) return -1;
  int32_t acc = 0;
  for (size_t i = 0; i < n; ++i) {
    int32_t t = i_apply(map_f, c, in0[i], in1 ? in1[i] : c);
    acc = (i == 0) ? t : i_apply(red_op, 0, acc, t);
  }
  *result = acc;
  return 0;
}

// ---- Scan (reading (c).4). inclusive: out[i] = x[0] (+) ... (+) x[i]; exclusive: out[0] = init,
// out[i] = init (+) x[0] (+) ... (+) x[i-1]. `out` may alias `x`.
void oracle_scan_i32(int op, int mode, int32_t init, const int32_t* x, size_t n, int32_t* out) {
  if (mode == SCAN_INCLUSIVE) {
    int32_t acc = 0;
    for (size_t i = 0; i < n; ++i) {
      acc = (i == 0) ? x[0] : i_apply(op, 0, acc, x[i]);
      out[i] = acc;
    }
  } else {
    int32_t acc = init;
    for (size_t i = 0; i < n; ++i) {
      int32_t xi = x[i];
      out[i] = acc;
      acc = i_apply(op, 0, acc, xi);
    }
  }
}

// fp32 scan in fp64 (plain running value, definition order); abs_prefix[i] = sum_{j<=i} |x[j]|
// (exclusive: |init| + sum_{j<i}) — the tolerance denominator of reading (c).4 v.
void oracle_scan_f32(int op, int mode, double init, const float* x, size_t n, double* out,
                     double* abs_prefix) {
  const double init32 = static_cast<double>(static_cast<float>(init));
  if (mode == SCAN_INCLUSIVE) {
    double acc = 0.0, aacc = 0.0;
    for (size_t i = 0; i < n; ++i) {
      acc = (i == 0) ? static_cast<double>(x[0]) : f_apply(op, 0.0, acc, x[i]);
      aacc += std::fabs(static_cast<double>(x[i]));
      out[i] = acc;
      if (abs_prefix) abs_prefix[i] = aacc;
    }
  } else {
    double acc = init32, aacc = std::fabs(init32);
    for (size_t i = 0; i < n; ++i) {
      double xi = x[i];
      out[i] = acc;
      if (abs_prefix) abs_prefix[i] = aacc;
      acc = f_apply(op, 0.0, acc, xi);
      aacc += std::fabs(xi);
    }
  }
}

// ---- MapOverlap 1D (reading (c).5) on a vector; outputs i in [i0, i1) into out[0 .. i1-i0).
// absout (optional) receives sum_k |w_k * x~_{i+k}|, the tolerance denominator.
void oracle_mapoverlap_1d_f32(const float* w, int r, int edge, double pad, const float* x, size_t n,
                              size_t i0, size_t i1, double* out, double* absout) {
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = static_cast<ptrdiff_t>(i0); i < static_cast<ptrdiff_t>(i1); ++i)
    overlap1_at(w, r, edge, pad, x, static_cast<ptrdiff_t>(n), 1, i, out + (i - i0),
                absout ? absout + (i - i0) : nullptr);
}

// the same applied along the rows (axis 0) or the columns (axis 1) of a row-major matrix; the
// f64 entry takes a fp64 input so the separable pair keeps its intermediate in fp64 ((c).6 iii)
void oracle_mapoverlap_1d_matrix_f32(const float* w, int r, int edge, double pad, int axis,
                                     const float* X, size_t rows, size_t cols, double* out,
                                     double* absout) {
  overlap1_matrix(w, r, edge, pad, axis, X, static_cast<ptrdiff_t>(rows), static_cast<ptrdiff_t>(cols), out, absout);
}
void oracle_mapoverlap_1d_matrix_f64(const float* w, int r, int edge, double pad, int axis,
                                     const double* X, size_t rows, size_t cols, double* out,
                                     double* absout) {
  overlap1_matrix(w, r, edge, pad, axis, X, static_cast<ptrdiff_t>(rows), static_cast<ptrdiff_t>(cols), out, absout);
}

// ---- MapOverlap 2D (reading (c).6); output rows [row0, row1) into out[0 .. (row1-row0)*cols).
void oracle_mapoverlap_2d_f32(const float* W, int ry, int rx, int edge, double pad, const float* X,
                              size_t rows, size_t cols, size_t row0, size_t row1, double* out,
                              double* absout) {
  overlap2_rows(W, ry, rx, edge, pad, X, static_cast<ptrdiff_t>(rows), static_cast<ptrdiff_t>(cols),
                static_cast<ptrdiff_t>(row0), static_cast<ptrdiff_t>(row1), out, absout);
}

// ---- int32 MapOverlap: 1D on a vector (outputs [i0, i1)), 1D along the rows / columns of a matrix, 2D
void oracle_mapoverlap_1d_i32(const int32_t* w, int r, int edge, int32_t pad, const int32_t* x, size_t n, size_t i0,
                              size_t i1, int32_t* out) {
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = static_cast<ptrdiff_t>(i0); i < static_cast<ptrdiff_t>(i1); ++i)
    out[i - i0] = ioverlap1_at(w, r, edge, pad, x, static_cast<ptrdiff_t>(n), 1, i);
}

void oracle_mapoverlap_1d_matrix_i32(const int32_t* w, int r, int edge, int32_t pad, int axis, const int32_t* X,
                                     size_t rows_, size_t cols_, int32_t* out) {
  const ptrdiff_t rows = static_cast<ptrdiff_t>(rows_), cols = static_cast<ptrdiff_t>(cols_);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < rows; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j)
      out[i * cols + j] = axis == AXIS_ROW ? ioverlap1_at(w, r, edge, pad, X + i * cols, cols, 1, j)
                                           : ioverlap1_at(w, r, edge, pad, X + j, rows, cols, i);
}

void oracle_mapoverlap_2d_i32(const int32_t* W, int ry, int rx, int edge, int32_t pad, const int32_t* X, size_t rows_,
                              size_t cols_, int32_t* out) {
  const ptrdiff_t rows = static_cast<ptrdiff_t>(rows_), cols = static_cast<ptrdiff_t>(cols_);
  const int fw = 2 * rx + 1;
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < rows; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j) {
      uint32_t acc = 0;
      for (int a = -ry; a <= ry; ++a)
        for (int b = -rx; b <= rx; ++b)
          acc += u32(W[(a + ry) * fw + (b + rx)]) * iext2(X, rows, cols, i + a, j + b, edge, pad);
      out[i * cols + j] = i32(acc);
    }
}

// ---- fp64 elements: every function returns the binary128 result rounded ONCE to fp64 -------------------------------
void oracle_map_f64(int fn, double c, const double* in0, const double* in1, size_t n, double* out) {
  const ptrdiff_t N = static_cast<ptrdiff_t>(n);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < N; ++i) out[i] = static_cast<double>(q_apply(fn, c, in0[i], in1 ? q128(in1[i]) : q128(c)));
}

void oracle_map3_f64(const double* in0, const double* in1, const double* in2, size_t n, double* out) {
  const ptrdiff_t N = static_cast<ptrdiff_t>(n);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < N; ++i) out[i] = static_cast<double>(q128(in0[i]) * q128(in1[i]) + q128(in2[i]));
}

int oracle_mapreduce_f64(int map_f /* -1: plain Reduce */, int red_op, double c, const double* in0, const double* in1,
                         size_t n, double* result, double* abs_sum) {
  if (n == 0) return -1;
  q128 acc = 0, aacc = 0;
  for (size_t i = 0; i < n; ++i) {
    const q128 t = map_f < 0 ? q128(in0[i]) : q_apply(map_f, c, in0[i], in1 ? q128(in1[i]) : q128(c));
    acc = i == 0 ? t : q_apply(red_op, 0, acc, t);
    aacc += q_abs(t);
  }
  *result = static_cast<double>(acc);
  if (abs_sum) *abs_sum = static_cast<double>(aacc);
  return 0;
}

void oracle_scan_f64(int op, int mode, double init, const double* x, size_t n, double* out, double* abs_prefix) {
  q128 acc = mode == SCAN_INCLUSIVE ? q128(0) : q128(init), aacc = mode == SCAN_INCLUSIVE ? q128(0) : q_abs(init);
  for (size_t i = 0; i < n; ++i) {
    if (mode == SCAN_INCLUSIVE) {
      acc = i == 0 ? q128(x[0]) : q_apply(op, 0, acc, x[i]);
      aacc += q_abs(x[i]);
      out[i] = static_cast<double>(acc);
      if (abs_prefix) abs_prefix[i] = static_cast<double>(aacc);
    } else {
      out[i] = static_cast<double>(acc);
      if (abs_prefix) abs_prefix[i] = static_cast<double>(aacc);
      acc = q_apply(op, 0, acc, x[i]);
      aacc += q_abs(x[i]);
    }
  }
}

void oracle_mapoverlap_1d_matrix_f64w(const double* w, int r, int edge, double pad, int axis, const double* X, size_t rows_,
                                      size_t cols_, double* out, double* absout) {
  const ptrdiff_t rows = static_cast<ptrdiff_t>(rows_), cols = static_cast<ptrdiff_t>(cols_);
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < rows; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j) {
      double* a = absout ? absout + i * cols + j : nullptr;
      if (axis == AXIS_ROW) qoverlap1_at(w, r, edge, pad, X + i * cols, cols, 1, j, out + i * cols + j, a);
      else qoverlap1_at(w, r, edge, pad, X + j, rows, cols, i, out + i * cols + j, a);
    }
}

void oracle_mapoverlap_2d_f64w(const double* W, int ry, int rx, int edge, double pad, const double* X, size_t rows_,
                               size_t cols_, double* out, double* absout) {
  const ptrdiff_t rows = static_cast<ptrdiff_t>(rows_), cols = static_cast<ptrdiff_t>(cols_);
  const int fw = 2 * rx + 1;
#pragma omp parallel for schedule(static)
  for (ptrdiff_t i = 0; i < rows; ++i)
    for (ptrdiff_t j = 0; j < cols; ++j) {
      q128 acc = 0, aacc = 0;
      for (int a = -ry; a <= ry; ++a)
        for (int b = -rx; b <= rx; ++b) {
          const q128 t = q128(W[(a + ry) * fw + (b + rx)]) * qext2(X, rows, cols, i + a, j + b, edge, pad);
          acc += t;
          aacc += q_abs(t);
        }
      out[i * cols + j] = static_cast<double>(acc);
      if (absout) absout[i * cols + j] = static_cast<double>(aacc);
    }
}

}  // extern "C"
