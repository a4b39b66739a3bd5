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

// Second probe: what a shared-memory load costs the FMA pipe. Every iteration issues 72 FFMA2 (144 FMA-pipe cycles per
// warp: the broadcast form of the stencil kernels, data register x uniform-register weight pair) and NL LDS.128 whose
// results are only XOR-ed together (ALU pipe). With NL = 0 the pipe runs at its peak; every LDS.128 takes ~4 cycles of
// it away (4 registers returned per thread: a saturated FMA pipe uses the whole register-file write bandwidth), which
// is what keeps the dense 9x9 MapOverlap at ~85 % of the FMA roofline however the rest is arranged.
struct alignas(16) ProbePairs { float2 p[16]; };
__device__ __forceinline__ unsigned long long probe_pack2(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
template <int NL>
__global__ void __launch_bounds__(PROBE_THREADS)
fma_lds_probe_kernel(const __grid_constant__ ProbePairs wp, const float* in, float* out, int iters) {
  __shared__ __align__(16) float sm[PROBE_THREADS * 4 * 8];
  for (int i = threadIdx.x; i < PROBE_THREADS * 4 * 8; i += PROBE_THREADS) sm[i] = in[i & 63];
  __syncthreads();
  float x[12], acc[16];
  unsigned junk = 0;
#pragma unroll
  for (int i = 0; i < 12; ++i) x[i] = in[(threadIdx.x + i) & 63];
#pragma unroll
  for (int i = 0; i < 16; ++i) acc[i] = 0.f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int l = 0; l < NL; ++l) {
      const uint4 t = *reinterpret_cast<const uint4*>(sm + threadIdx.x * 4 + ((it + l) & 7) * (PROBE_THREADS * 4));
      junk ^= t.x ^ t.y ^ t.z ^ t.w;
    }
#pragma unroll
    for (int o = 0; o < 4; ++o)
#pragma unroll
      for (int d = 0; d < 9; ++d)
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          unsigned long long r;
          asm("fma.rn.f32x2 %0, %1, %2, %3;"
              : "=l"(r)
              : "l"(probe_pack2(x[d + 2 * q], x[d + 2 * q])), "l"(probe_pack2(wp.p[d + o].x, wp.p[d + o].y)),
                "l"(probe_pack2(acc[4 * o + 2 * q], acc[4 * o + 2 * q + 1])));
          asm("mov.b64 {%0, %1}, %2;" : "=f"(acc[4 * o + 2 * q]), "=f"(acc[4 * o + 2 * q + 1]) : "l"(r));
        }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += acc[i];
  if (s == 123.456f || junk == 0x12345u) out[0] = s;
}

}  // namespace

cudaError_t launch_fma_lds_probe(const Launch& L, int nl, const float* in64, float* scratch, double* fma_count) {
  ProbePairs wp;
  for (int i = 0; i < 16; ++i) wp.p[i] = make_float2(1e-3f * i, 2e-3f * i);
  const unsigned grid = unsigned(L.sms) * 3;  // three resident blocks per SM, like the 9x9 kernel
  const int iters = 2000;
  switch (nl) {
    case 0: fma_lds_probe_kernel<0><<<grid, PROBE_THREADS, 0, L.stream>>>(wp, in64, scratch, iters); break;
    case 1: fma_lds_probe_kernel<1><<<grid, PROBE_THREADS, 0, L.stream>>>(wp, in64, scratch, iters); break;
    case 2: fma_lds_probe_kernel<2><<<grid, PROBE_THREADS, 0, L.stream>>>(wp, in64, scratch, iters); break;
    case 4: fma_lds_probe_kernel<4><<<grid, PROBE_THREADS, 0, L.stream>>>(wp, in64, scratch, iters); break;
    case 8: fma_lds_probe_kernel<8><<<grid, PROBE_THREADS, 0, L.stream>>>(wp, in64, scratch, iters); break;
    default: return cudaErrorInvalidValue;
  }
  ++*L.launches;
  *fma_count = double(grid) * PROBE_THREADS * double(iters) * 144.0;
  return cudaGetLastError();
}

cudaError_t launch_fma_probe(const Launch& L, float* scratch, double* fma_count) {
  const unsigned grid = unsigned(L.sms) * 8;
  fma_probe_kernel<<<grid, PROBE_THREADS, 0, L.stream>>>(scratch, 0.999f, 0.001f);
  ++*L.launches;
  *fma_count = double(grid) * PROBE_THREADS * double(PROBE_ITERS) * PROBE_CHAINS;
  return cudaGetLastError();
}

}  // namespace skel
