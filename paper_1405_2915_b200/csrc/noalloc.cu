// Reduce for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): skel_reduce_f32_noalloc (include/skel.h). The Reduce of reduce.cu (one block per contiguous chunk, one
// partial per block, the block that draws the last ticket folds the partials in index order) with its scratch - the
// partials and the ticket - in a file-scope __device__ array instead of the context's cudaMalloc'ed scratch.
//
//   * The array costs NOALLOC_SCRATCH_BYTES (33 024 B) on every GPU that loads the library, until the process exits.
//   * At most NOALLOC_MAX_ELEMENTS = 2^26 elements per call (8192 chunks of 8192 elements); more is rejected.
//   * Every call shares the array: calls that overlap on the GPU (two streams, two host threads) race on the partials
//     and on the ticket. Calls on one stream are ordered and safe. The ticket is cleared on the stream before every
//     launch, so a call that was cut short cannot poison the next one; the partials need no clearing (every slot that
//     is read was written by this launch).
//   * The entry point calls no cudaMalloc / cudaFree / allocating library routine: cudaGetDevice, once per device
//     cudaGetSymbolAddress (the array's name is a HOST-side stand-in in host code, not a device address), then
//     cudaMemsetAsync (4 bytes) and the kernel launch.
#include "common.cuh"
#include "kernels.hpp"
#include "../../include/skel.h"
#include <mutex>
#include <stdio.h>

namespace skel {
namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_V = 4, NA_U = 4;                                    // 128-bit loads, four per thread in flight
constexpr size_t NA_TILE = size_t(NA_THREADS) * NA_V * NA_U;         // 4096 elements
constexpr size_t NA_CHUNK = 2 * NA_TILE;                             // 8192 elements = 32 KB per block
constexpr size_t NA_MAX_BLOCKS = 8192;
constexpr size_t NOALLOC_MAX_ELEMENTS = NA_MAX_BLOCKS * NA_CHUNK;    // 2^26
constexpr size_t NA_TICKET_OFFSET = NA_MAX_BLOCKS * sizeof(float);   // 32 768, a multiple of 256
constexpr size_t NOALLOC_SCRATCH_BYTES = NA_TICKET_OFFSET + 256;

// partials[8192] (float), then the ticket (unsigned) in a 256-byte line of its own
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

template <int OP>
__global__ void __launch_bounds__(NA_THREADS)
reduce_noalloc_kernel(const float* in, size_t n, unsigned char* scratch, float* result) {
  __shared__ float smem[32];
  __shared__ bool is_last;
  float* partials = reinterpret_cast<float*>(scratch);
  unsigned* ticket = reinterpret_cast<unsigned*>(scratch + NA_TICKET_OFFSET);
  const bool vec_ok = reinterpret_cast<uintptr_t>(in) % 16 == 0;
  float acc[NA_V];
#pragma unroll
  for (int j = 0; j < NA_V; ++j) acc[j] = identity<float, OP>();
  const size_t lo = size_t(blockIdx.x) * NA_CHUNK;
#pragma unroll 1
  for (size_t tile = lo; tile < lo + NA_CHUNK && tile < n; tile += NA_TILE) {
    const size_t base = tile + size_t(threadIdx.x) * NA_V;
    if (vec_ok && tile + NA_TILE <= n) {
      uint32_t a[NA_U][NA_V];
#pragma unroll
      for (int u = 0; u < NA_U; ++u) ld_stream<NA_V, true>(a[u], in + base + size_t(u) * NA_THREADS * NA_V);
#pragma unroll
      for (int u = 0; u < NA_U; ++u)
#pragma unroll
        for (int j = 0; j < NA_V; ++j) acc[j] = apply_fn<OP>(0.f, acc[j], __uint_as_float(a[u][j]));
    } else {
#pragma unroll
      for (int u = 0; u < NA_U; ++u)
#pragma unroll
        for (int j = 0; j < NA_V; ++j) {
          const size_t i = base + size_t(u) * NA_THREADS * NA_V + j;
          if (i < n) acc[j] = apply_fn<OP>(0.f, acc[j], in[i]);
        }
    }
  }
  float v = acc[0];
#pragma unroll
  for (int j = 1; j < NA_V; ++j) v = apply_fn<OP>(0.f, v, acc[j]);
  v = block_reduce<float, OP>(v, smem);
  if (gridDim.x == 1) {
    if (threadIdx.x == 0) *result = v;
    return;
  }
  if (threadIdx.x == 0) {
    partials[blockIdx.x] = v;
    __threadfence();
    is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (is_last) {
    __threadfence();
    float a = identity<float, OP>();
    for (unsigned k = threadIdx.x; k < gridDim.x; k += NA_THREADS) a = apply_fn<OP>(0.f, a, partials[k]);
    __syncthreads();  // smem reuse
    a = block_reduce<float, OP>(a, smem);
    if (threadIdx.x == 0) *result = a;
  }
}

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_addr[NA_MAX_DEVICES];  // device address of g_noalloc_scratch on each device, once resolved
thread_local char g_noalloc_error[256] = "";

skel_status fail(skel_status s, const char* fmt, const char* detail = "", unsigned long long a = 0, unsigned long long b = 0) {
  snprintf(g_noalloc_error, sizeof g_noalloc_error, fmt, detail, a, b);
  return s;
}

// set-up, once per device, with that device current
skel_status scratch_for_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(SKEL_ERR_CUDA, "skel_reduce_f32_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(SKEL_ERR_UNSUPPORTED, "skel_reduce_f32_noalloc: device ordinal out of range%s");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_addr[dev]) {
    unsigned char* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_noalloc_scratch);
    if (e != cudaSuccess || !p)
      return fail(SKEL_ERR_CUDA, "skel_reduce_f32_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return SKEL_OK;
}

}  // namespace
}  // namespace skel

#pragma GCC visibility push(default)
extern "C" {

size_t skel_noalloc_max_elements(void) { return skel::NOALLOC_MAX_ELEMENTS; }
size_t skel_noalloc_scratch_bytes(void) { return skel::NOALLOC_SCRATCH_BYTES; }
const char* skel_noalloc_last_error(void) { return skel::g_noalloc_error; }

skel_status skel_reduce_f32_noalloc(skel_fn op, const float* device_in, size_t n, float* device_result, void* cuda_stream) {
  using namespace skel;
  if (!device_in || !device_result) return fail(SKEL_ERR_INVALID_ARG, "skel_reduce_f32_noalloc: NULL pointer%s");
  if (op != SKEL_FN_ADD && op != SKEL_FN_MULT && op != SKEL_FN_MAX)
    return fail(SKEL_ERR_INVALID_ARG, "skel_reduce_f32_noalloc: op must be ADD, MULT or MAX%s");
  if (n == 0) return fail(SKEL_ERR_EMPTY, "skel_reduce_f32_noalloc: n == 0 (no identity is passed)%s");
  if (n > NOALLOC_MAX_ELEMENTS)
    return fail(SKEL_ERR_UNSUPPORTED, "skel_reduce_f32_noalloc:%s n = %llu exceeds the static scratch's maximum of %llu elements",
                "", (unsigned long long)n, (unsigned long long)NOALLOC_MAX_ELEMENTS);
  unsigned char* scratch = nullptr;
  const skel_status s = scratch_for_current_device(&scratch);
  if (s != SKEL_OK) return s;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const unsigned grid = static_cast<unsigned>((n + NA_CHUNK - 1) / NA_CHUNK);
  cudaError_t e = cudaSuccess;
  if (grid > 1) e = cudaMemsetAsync(scratch + NA_TICKET_OFFSET, 0, sizeof(unsigned), stream);  // the ticket starts at zero
  if (e == cudaSuccess) {
    if (op == SKEL_FN_ADD) reduce_noalloc_kernel<FN_ADD><<<grid, NA_THREADS, 0, stream>>>(device_in, n, scratch, device_result);
    else if (op == SKEL_FN_MULT) reduce_noalloc_kernel<FN_MULT><<<grid, NA_THREADS, 0, stream>>>(device_in, n, scratch, device_result);
    else reduce_noalloc_kernel<FN_MAX><<<grid, NA_THREADS, 0, stream>>>(device_in, n, scratch, device_result);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return fail(SKEL_ERR_CUDA, "skel_reduce_f32_noalloc: %s", cudaGetErrorString(e));
  g_noalloc_error[0] = 0;
  return SKEL_OK;
}

}  // extern "C"
#pragma GCC visibility pop
