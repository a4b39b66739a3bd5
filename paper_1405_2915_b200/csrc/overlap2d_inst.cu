// One instantiation set of the tiled MapOverlap 2D / column-wise kernels (overlap2d_tiles.cuh).
// Compiled once per value of SKEL_INST (build.py): 0..3 = dense 2D with ry = rx = 1..4;
// 4..9 = column-wise 1D with r = 1, 2, 3, 4, 8, 16.
#include "overlap2d_tiles.cuh"

#ifndef SKEL_INST
#error "compile with -DSKEL_INST=<0..9>"
#endif

namespace skel {

#define SKEL_DEF_2D(R)                                                                                              \
  template <>                                                                                                       \
  cudaError_t launch_overlap2d_tiled<R>(const Launch& L, int v, int dtype, const Weights2D& w, int edge, float pad, \
                                        const float* in, float* out, size_t rows, size_t cols) {                    \
    return launch_tiled_any<R, R, Weights2D>(L, v, dtype, w, edge, pad, in, out, rows, cols);                       \
  }
#define SKEL_DEF_COL(R)                                                                                             \
  template <>                                                                                                       \
  cudaError_t launch_overlap1d_cols_tiled<R>(const Launch& L, int v, int dtype, const Weights1D& w, int edge,       \
                                             float pad, const float* in, float* out, size_t rows, size_t cols) {    \
    return launch_tiled_any<R, 0, Weights1D>(L, v, dtype, w, edge, pad, in, out, rows, cols);                       \
  }

#if SKEL_INST == 0
SKEL_DEF_2D(1)
#elif SKEL_INST == 1
SKEL_DEF_2D(2)
#elif SKEL_INST == 2
SKEL_DEF_2D(3)
#elif SKEL_INST == 3
SKEL_DEF_2D(4)
#elif SKEL_INST == 4
SKEL_DEF_COL(1)
#elif SKEL_INST == 5
SKEL_DEF_COL(2)
#elif SKEL_INST == 6
SKEL_DEF_COL(3)
#elif SKEL_INST == 7
SKEL_DEF_COL(4)
#elif SKEL_INST == 8
SKEL_DEF_COL(8)
#elif SKEL_INST == 9
SKEL_DEF_COL(16)
#else
#error "SKEL_INST out of range"
#endif

}  // namespace skel
