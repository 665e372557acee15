// launch_cfg.h — one-time, per-device, thread-safe launch configuration shared by the tuned kernels' launchers:
// the opt-in to more than 48 KB of dynamic shared memory (cudaFuncSetAttribute is per function AND per device) and the
// SM count of the current device. A second device or a second host thread in the same process gets its own entries.
#ifndef SC_LAUNCH_CFG_H_
#define SC_LAUNCH_CFG_H_

#include <cuda_runtime.h>

#include <map>
#include <mutex>
#include <utility>

namespace sc {

inline int current_device() {
  int d = 0;
  if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); d = 0; }
  return d;
}

inline int device_sm_count() {
  static std::mutex mu;
  static std::map<int, int> cache;
  const int dev = current_device();
  std::lock_guard<std::mutex> g(mu);
  auto it = cache.find(dev);
  if (it != cache.end()) return it->second;
  int n = 148;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); n = 148; }
  cache[dev] = n;
  return n;
}

// make `bytes` of dynamic shared memory available to `kernel` on the current device (idempotent, grows only)
template <class Kernel>
inline cudaError_t ensure_dynamic_smem(Kernel kernel, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<const void*, int>, size_t> done;
  const std::pair<const void*, int> key(reinterpret_cast<const void*>(kernel), current_device());
  std::lock_guard<std::mutex> g(mu);
  auto it = done.find(key);
  if (it != done.end() && it->second >= bytes) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) done[key] = bytes;
  return e;
}

}  // namespace sc
#endif
