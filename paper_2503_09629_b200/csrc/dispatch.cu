// dispatch.cu — picks the kernel set: the tuned sm_100a kernels (default: stage_tma.cu, ghost_tiled.cu,
// restrict_zmarch.cu) or the straightforward direct-load kernels of kernels_basic.cu (environment
// SC_KERNELS=ref; A/B checks and debugging only). Both are CUDA; there is no CPU path.
#include "kernels.h"

namespace sc {

void launch_stage_direct(const StageArgs& a, cudaStream_t st);
void launch_stage_tma(const StageArgs& a, cudaStream_t st);
bool make_box_tensor_map_tma(const BoxView& b, int narrays, void* base, void* out_map128);
void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st);
void launch_ghost_fill_tiled(const GhostArgs& a, cudaStream_t st);
void launch_restrict_ref(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);
void launch_restrict_opt(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);

static int g_mode = 1;
void select_kernels(int mode) { g_mode = mode; }
int selected_kernels() { return g_mode; }

void launch_stage(const StageArgs& a, cudaStream_t st) {
  if (g_mode == 0) launch_stage_direct(a, st);
  else launch_stage_tma(a, st);
}
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st) {
  if (g_mode == 0 || a.ntiles == 0) launch_ghost_fill_direct(a, st);
  else launch_ghost_fill_tiled(a, st);
}
void launch_restrict(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st) {
  if (g_mode == 0) launch_restrict_ref(ch, pa, V, yc, yp, st);
  else launch_restrict_opt(ch, pa, V, yc, yp, st);
}
bool make_box_tensor_map(const BoxView& b, int narrays, void* base, void* out_map128) {
  return make_box_tensor_map_tma(b, narrays, base, out_map128);
}

}  // namespace sc
