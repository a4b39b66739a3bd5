// FP32 FMA roofline probe ("the FMA roofline is to be measured by a register-only FFMA
// micro-benchmark in the same run"): every thread runs ITERS x 16 independent fused multiply-adds on
// registers; the grid fills every SM with 8 blocks of 256 threads. Used by bench.py to report the
// arithmetic-bound MapOverlap rows (dense 9x9, 1D r = 16) against the FP32 pipe instead of HBM.
#include "common.cuh"
#include "kernels.hpp"

namespace skel {
namespace {

constexpr int PROBE_ITERS = 4096, PROBE_CHAINS = 16, PROBE_THREADS = 256;

__global__ void __launch_bounds__(PROBE_THREADS) fma_probe_kernel(float* out, float a, float b) {
  float acc[PROBE_CHAINS];
#pragma unroll
  for (int i = 0; i < PROBE_CHAINS; ++i) acc[i] = threadIdx.x * 0.001f + i;
  for (int it = 0; it < PROBE_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PROBE_CHAINS; ++i) acc[i] = fmaf(acc[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PROBE_CHAINS; ++i) s += acc[i];
  if (s == 123.456f) out[0] = s;  // never true for the arguments used: keeps the loop alive
}

}  // namespace

cudaError_t launch_fma_probe(const Launch& L, float* scratch, double* fma_count) {
  const unsigned grid = unsigned(L.sms) * 8;
  fma_probe_kernel<<<grid, PROBE_THREADS, 0, L.stream>>>(scratch, 0.999f, 0.001f);
  ++*L.launches;
  *fma_count = double(grid) * PROBE_THREADS * double(PROBE_ITERS) * PROBE_CHAINS;
  return cudaGetLastError();
}

}  // namespace skel
