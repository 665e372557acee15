// noalloc.cu — sc_max_abs_noalloc: the blow-up check of sc_debug_max_abs for callers that must not allocate.
//
// Who this is for. sc_debug_max_abs needs a hierarchy, and sc_create_hierarchy calls cudaMalloc (staging buffer, tile
// lists) even when the caller brings its own arena. Two kinds of caller cannot afford that:
//   - a host application that has handed ALL device memory to its own pool at start-up (AMR drivers and ML frameworks
//     both do this): a cudaMalloc from a library then simply fails with out-of-memory, however small the request;
//   - a time loop that watches a running simulation for NaN / inf every few steps: cudaMalloc and cudaFree
//     synchronise the whole device, so a monitor that allocates stalls every stream of the application.
// For them this file offers one call that takes the caller's input and output pointers and touches no allocator at
// all: no cudaMalloc / cudaFree / cudaMallocAsync, no library routine that allocates.
//
// How. The reduction needs a little global memory that is neither input nor output (one partial maximum per thread
// block and an arrival counter). It lives in a file-scope __device__ array of fixed size, which the CUDA runtime places
// on every GPU that loads libsubcycle.so and keeps there until the process exits (about 64 KB per GPU). The price is a
// hard limit on the input length, SC_NOALLOC_MAX_DOUBLES, checked on entry.
//
// Sharing. There is ONE such array per GPU and every call on that GPU uses it. It still holds the previous call's
// partials when the next call starts; the call therefore clears the arrival counter on the stream before the kernel,
// and the kernel reads back only the partials its own blocks wrote. Two calls whose kernels can overlap on the same
// GPU (different streams, or different host threads on different streams) race on the array and both results are
// garbage: keep all calls for one GPU on one stream, or order them with events.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "../../include/subcycle.h"
#include "sc_internal.h"

namespace sc {
namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CHUNK = 8192;                                    // doubles reduced by one thread block
constexpr int NA_MAX_BLOCKS = (int)(SC_NOALLOC_MAX_DOUBLES / NA_CHUNK);
constexpr int NA_HEADER = 32;                                     // 256 bytes: word 0 = arrival counter, rest unused
static_assert((unsigned long long)NA_MAX_BLOCKS * NA_CHUNK == SC_NOALLOC_MAX_DOUBLES, "limit must be whole chunks");

// The scratch itself. In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address and
// must never be passed to a kernel as a pointer (the kernel would fault, or on machines where the GPU can read host
// memory, quietly work on the wrong bytes). Host code below always goes through scratch_for_current_device().
static __device__ __align__(256) unsigned long long noalloc_scratch[NA_HEADER + NA_MAX_BLOCKS];

constexpr int NA_MAX_DEVICES = 64;
std::mutex na_mu;
unsigned long long* na_addr[NA_MAX_DEVICES] = {};  // device address of noalloc_scratch on GPU d, resolved once

// One-time set-up per GPU: ask the runtime where noalloc_scratch lives on the CURRENT device. Each GPU has its own copy
// at its own address, so the answer is cached per device ordinal and must be looked up with that device current.
cudaError_t scratch_for_current_device(unsigned long long** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> g(na_mu);
  if (!na_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, noalloc_scratch);
    if (e != cudaSuccess) return e;
    na_addr[dev] = static_cast<unsigned long long*>(p);
  }
  *out = na_addr[dev];
  return cudaSuccess;
}

__device__ inline unsigned long long umax64(unsigned long long a, unsigned long long b) { return a > b ? a : b; }

// maximum over the block; valid in thread 0
__device__ inline unsigned long long block_max(unsigned long long m, unsigned long long* sh) {
  for (int s = 16; s > 0; s >>= 1) m = umax64(m, __shfl_xor_sync(0xffffffffu, m, s));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    m = threadIdx.x < NA_THREADS / 32 ? sh[threadIdx.x] : 0ull;
    for (int s = 16; s > 0; s >>= 1) m = umax64(m, __shfl_xor_sync(0xffffffffu, m, s));
  }
  __syncthreads();
  return m;
}

// Same ordering trick as max_abs_kernel (kernels_basic.cu): |x| of a NaN has a larger bit pattern than +inf, which has
// a larger one than any finite magnitude, so the unsigned maximum of the bit patterns of |x| is NaN if there is one,
// else +inf if there is one, else the largest magnitude. Block b reduces x[b*NA_CHUNK, (b+1)*NA_CHUNK) and stores its
// partial; the block that arrives last folds the gridDim.x partials of THIS launch and writes *out.
__global__ void __launch_bounds__(NA_THREADS) max_abs_noalloc_kernel(const double* __restrict__ x, unsigned long long n,
                                                                     double* __restrict__ out,
                                                                     unsigned long long* __restrict__ scratch) {
  __shared__ unsigned long long sh[NA_THREADS / 32];
  __shared__ bool last;
  unsigned long long* partial = scratch + NA_HEADER;
  const unsigned long long lo = (unsigned long long)blockIdx.x * NA_CHUNK;
  const unsigned long long hi = lo + NA_CHUNK < n ? lo + NA_CHUNK : n;
  unsigned long long m = 0ull;
  for (unsigned long long i = lo + threadIdx.x; i < hi; i += NA_THREADS)
    m = umax64(m, (unsigned long long)__double_as_longlong(fabs(x[i])));
  m = block_max(m, sh);
  if (threadIdx.x == 0) {
    partial[blockIdx.x] = m;
    __threadfence();  // the partial is visible before the arrival is counted
    last = atomicAdd(scratch, 1ull) == (unsigned long long)gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  m = 0ull;
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += NA_THREADS) m = umax64(m, __ldcg(partial + b));
  m = block_max(m, sh);
  if (threadIdx.x == 0) *out = __longlong_as_double((long long)m);
}

}  // namespace
}  // namespace sc

extern "C" int32_t sc_max_abs_noalloc(const double* x, uint64_t n, double* out, void* cuda_stream) {
  using namespace sc;
  if (!out) { set_error("sc_max_abs_noalloc: null out"); return SC_ERR_INVALID_ARG; }
  if (!x && n) { set_error("sc_max_abs_noalloc: null x"); return SC_ERR_INVALID_ARG; }
  if (n > SC_NOALLOC_MAX_DOUBLES) {
    set_error("sc_max_abs_noalloc: n = " + std::to_string(n) + " doubles exceeds SC_NOALLOC_MAX_DOUBLES = " +
              std::to_string((unsigned long long)SC_NOALLOC_MAX_DOUBLES) +
              " (the size of the built-in scratch array); split the input and combine the maxima");
    return SC_ERR_INVALID_ARG;
  }
  unsigned long long* scratch = nullptr;
  cudaError_t e = scratch_for_current_device(&scratch);
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_error(std::string("sc_max_abs_noalloc: cudaGetSymbolAddress of the scratch array: ") + cudaGetErrorString(e));
    return SC_ERR_CUDA;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // the arrival counter must start at zero whatever an earlier (possibly aborted) call left behind
  e = cudaMemsetAsync(scratch, 0, NA_HEADER * sizeof(unsigned long long), st);
  if (e == cudaSuccess) {
    const unsigned nblocks = n ? (unsigned)((n + NA_CHUNK - 1) / NA_CHUNK) : 1u;
    max_abs_noalloc_kernel<<<nblocks, NA_THREADS, 0, st>>>(x, (unsigned long long)n, out, scratch);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    set_error(std::string("sc_max_abs_noalloc: ") + cudaGetErrorString(e));
    return SC_ERR_CUDA;
  }
  return SC_OK;
}
