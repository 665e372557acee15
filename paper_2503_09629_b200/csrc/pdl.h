// pdl.h — programmatic dependent launch (sm_90+) for the step's kernel chain. A coarse step is a strictly serial
// chain of 200-1000 short kernels (15-170 us each). The tuned kernels are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization (captured into the CUDA graph as programmatic edges) and
// start with pdl_enter() = griddepcontrol.wait, which returns once the previous grid has COMPLETED and its writes
// are visible — the full dependency; nothing is read or written before it. No kernel issues
// griddepcontrol.launch_dependents: the dependent grid is released when the previous grid's last CTA exits, so
// only its launch processing overlaps the previous kernel's teardown. Measured (profiles/r01_v4.md): cfg 5
// 21.76 -> 21.64 ms, cfg 3 0.807 -> 0.802 ms per coarse step. Releasing the dependents EARLIER (at the top of every
// kernel, or when a CTA starts its last planes / last item) was slower in every variant tried (22.0-22.8 ms;
// cfg 3 0.834 ms): the early CTAs land on whichever SMs drain first and the next kernel starts unbalanced.
// A kernel launched through launch_pdl() MUST call pdl_enter() before touching global memory. SC_PDL=0 in the
// environment launches everything without the attribute (A/B checks).
#ifndef SC_PDL_H_
#define SC_PDL_H_

#include <cuda_runtime.h>

#include <cstdlib>
#include <utility>

namespace sc {

__device__ __forceinline__ void pdl_enter() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

inline bool pdl_enabled() {
  static const bool on = [] {
    const char* e = getenv("SC_PDL");
    return !(e && e[0] == '0');
  }();
  return on;
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl_enabled() ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

}  // namespace sc
#endif
